"""GPU: the no-allocation entry point pimd_row_scan_noalloc_dev (include/pimd_noalloc.h) against the existing path.

The existing path is the row-index scan the context runs inside every force evaluation (scratch from the context's
arena), read back with pimd_debug_get_row_index.  Integer work: the bar is bit-exact.  The file sorts last on purpose
(pytest -x: a failure here must not hide another test) and passes alone in a fresh process as well
as after the other tests -- it keeps no state besides the library's static scratch, which every call rewrites.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _context_row_index(k):
    """(n_types, cen_idx, ncount, rowstart) of configs[k]'s initial force evaluation, from the context's own path."""
    import paper_2602_13553_b200 as pk
    import workloads
    cfg, wb, desc, w = workloads.make_config(k)
    sim = pk.PIMD(wb["types"], wb["masses"], wb["box"], cfg["P"], cfg["T"], cfg["dt"], cfg["gamma"], seed=3, model_desc=desc)
    sim.set_state(wb["x"], wb["p"])
    sim.set_model(w)
    nt = len(wb["masses"])
    ncount = pk.pimd_get_neighbor_counts(sim.ctx, sim.P, sim.N, nt).reshape(sim.P * sim.N, nt)
    cen, rowstart = pk.pimd_debug_get_row_index(sim.ctx, sim.P, sim.N, nt)
    sim.close()
    return nt, cen, ncount, rowstart


def _plain_scan(nt, cen, ncount):
    """the definition in pimd_noalloc.h written out (an independent check of both paths)"""
    out = np.zeros((nt, cen.size + 1), dtype=np.int64)
    for tj in range(nt):
        out[tj, 1:] = np.cumsum(ncount[cen, tj].astype(np.int64))
    return out


def test_row_scan_noalloc_equals_the_context_path_on_two_calls_in_a_row():
    import torch
    import paper_2602_13553_b200 as pk
    pk.pimd_noalloc_setup()
    big = _context_row_index(1)        # 192 atoms x 32 beads = 6144 centres: 6 scan blocks and a ragged tail of warps
    small = _context_row_index(0)      # 96 x 4 = 384 centres: one partial block
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream(dev).cuda_stream
    # two calls in a row, the larger first so that the smaller one finds its block sums and everything behind them stale,
    # then the larger again over the smaller one's left-overs
    free_before = None
    for nt, cen, ncount, rowstart in (big, small, big):
        assert np.array_equal(rowstart.astype(np.int64), _plain_scan(nt, cen, ncount))
        cen_d = torch.from_numpy(cen).to(dev)
        cnt_d = torch.from_numpy(np.ascontiguousarray(ncount)).to(dev)
        out_d = torch.full((nt, cen.size + 1), -7, dtype=torch.int32, device=dev)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(dev)[0]
        pk.pimd_row_scan_noalloc_dev(cen.size, nt, cen_d, cnt_d, out_d, stream)
        pk.pimd_row_scan_noalloc_dev(cen.size, nt, cen_d, cnt_d, out_d, stream)      # and once more on the same buffers
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info(dev)[0] == free_before                        # the call took no device memory
        assert np.array_equal(out_d.cpu().numpy(), rowstart)                         # bit-exact with the context's path


def test_row_scan_noalloc_refuses_sizes_beyond_its_scratch():
    import torch
    import paper_2602_13553_b200 as pk
    dev = torch.device("cuda:0")
    one = torch.zeros(8, dtype=torch.int32, device=dev)
    for n_centres, n_types, word in ((4194304 + 1, 2, "PIMD_NOALLOC_MAX_CENTRES"), (4, 5, "n_types"), (0, 2, "n_centres")):
        with pytest.raises(pk.PimdError) as ei:
            pk.pimd_row_scan_noalloc_dev(n_centres, n_types, one.data_ptr(), one.data_ptr(), one.data_ptr())
        assert ei.value.code == pk.PIMD_EINVAL and word in str(ei.value)
    with pytest.raises(pk.PimdError):
        pk.pimd_row_scan_noalloc_dev(4, 2, 0, one.data_ptr(), one.data_ptr())
    torch.cuda.synchronize()
    # the largest size the scratch admits runs (4096 scan blocks x 2 types): every centre one neighbour of each type
    n = 4194304
    cen = torch.arange(n, dtype=torch.int32, device=dev)
    cnt = torch.ones((n, 2), dtype=torch.int32, device=dev)
    out = torch.empty((2, n + 1), dtype=torch.int32, device=dev)
    pk.pimd_row_scan_noalloc_dev(n, 2, cen, cnt, out)
    torch.cuda.synchronize()
    want = torch.arange(n + 1, dtype=torch.int32, device=dev)
    assert torch.equal(out[0], want) and torch.equal(out[1], want)
