// neighbor.cu -- F1 (wrap + per-bead cell binning) and F2 (neighbour rows + smooth environment matrix)
// of SURVEY 8(a).  Geometry is FP64 with the exact operation order of DESIGN R-11 (no FMA
// contraction: __dmul_rn / __dadd_rn), so the neighbour sets are bit-identical to the oracle's.
//   w = x - L*floor(x/L)                                   PAPER.md:L200-202 (wrap before the force call)
//   rows (j, n): d = (w_j - w_i) + n*L,  (dx^2+dy^2)+dz^2 < rc^2 strictly, (j,n) != (i,0)    R-11
//   s(r) smooth switch, R_row = (s, s d/r)                 R-12
// All images are enumerated (box may be shorter than 2 r_c: configs[0]), by walking cell offsets
// -R..R with R = ceil(r_c / cell width) and recording the lattice shift n of every wrap-around.
#include "common.cuh"

namespace pimd {

struct GridGeom {
    double L[3];
    double inv_w[3];     // ncell / L
    double cw[3];        // cell width L / ncell
    double inv_nc[3];    // 1 / ncell
    int nc[3];
    int R[3];
    int ncells;
    const double* boxp;  // barostat (PAPER.md Eq. E6): the cell is rescaled on the device every step; null = use L
    double rc;
    int* overflow;
    long long* ctl;      // device step counter of the graph-replayed step loop (api.cu): advanced once per evaluation
};

// cell lengths and inverse cell widths of this launch: kernel arguments, or the device-resident cell under a barostat
__device__ __forceinline__ void load_geom(const GridGeom& g, double L[3], double inv_w[3]) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        L[a] = g.boxp ? g.boxp[a] : g.L[a];
        inv_w[a] = g.boxp ? (double)g.nc[a] / L[a] : g.inv_w[a];
    }
}
// cell widths (only the pruning test uses them: its 1e-6 margin dwarfs the rounding of L * (1/nc))
__device__ __forceinline__ void load_widths(const GridGeom& g, const double L[3], double cw[3]) {
#pragma unroll
    for (int a = 0; a < 3; ++a) cw[a] = g.boxp ? L[a] * g.inv_nc[a] : g.cw[a];
}

__global__ void wrap_bin_kernel(int P, int N, GridGeom g, const double* __restrict__ x, double* __restrict__ wtmp,
                                int* __restrict__ cell_id, int* __restrict__ cell_count) {
    const int ba = blockIdx.x * blockDim.x + threadIdx.x;
    if (ba >= P * N) return;
    const int k = ba / N;
    double gL[3], ginv_w[3];
    load_geom(g, gL, ginv_w);
    if (ba == 0) {
        const int ev = g.overflow[2] + 1;            // force evaluations since pimd_set_model, this one included
        g.overflow[2] = ev;
        if (g.ctl) g.ctl[0] += 1;                    // the next integrator launch opens the next step
        if (g.boxp) {
            // the cell shrank so far inside one pimd_step call that rc spans more than R cells: neighbours would be missed
            for (int a = 0; a < 3; ++a)
                if (g.rc * ginv_w[a] > (double)g.R[a]) {
                    atomicOr(g.overflow, 2);
                    atomicMin(reinterpret_cast<unsigned*>(g.overflow) + 1, (unsigned)ev);
                }
        }
    }
    int c[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double xv = x[(size_t)ba * 3 + a];
        const double w = __dsub_rn(xv, __dmul_rn(gL[a], floor(__ddiv_rn(xv, gL[a]))));
        wtmp[(size_t)ba * 3 + a] = w;
        int ci = (int)floor(w * ginv_w[a]);
        ci = ci < 0 ? 0 : (ci >= g.nc[a] ? g.nc[a] - 1 : ci);
        c[a] = ci;
    }
    const int cid = (c[2] * g.nc[1] + c[1]) * g.nc[0] + c[0];
    cell_id[ba] = cid;
    atomicAdd(cell_count + (size_t)k * (g.ncells + 1) + cid, 1);
}

// exclusive scan of the cell counts of one bead (one block per bead)
__global__ void cell_scan_kernel(int ncells, const int* __restrict__ cell_count, int* __restrict__ cell_start) {
    __shared__ int warp_tot[32];
    __shared__ int carry;
    const int k = blockIdx.x;
    const int* cnt = cell_count + (size_t)k * (ncells + 1);
    int* start = cell_start + (size_t)k * (ncells + 1);
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < ncells + 1; base += blockDim.x) {
        const int idx = base + threadIdx.x;
        const int v = (idx < ncells) ? cnt[idx] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if ((threadIdx.x & 31) >= o) incl += t;
        }
        if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = incl;
        __syncthreads();
        int woff = 0;
        for (int q = 0; q < (int)(threadIdx.x >> 5); ++q) woff += warp_tot[q];
        const int excl = carry + woff + incl - v;
        if (idx < ncells + 1) start[idx] = excl;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = excl + v;
        __syncthreads();
    }
}

__global__ void cell_fill_kernel(int P, int N, int ncells, const int* __restrict__ cell_id,
                                 const int* __restrict__ cell_start, int* __restrict__ cell_fill,
                                 int* __restrict__ cell_tmp) {
    const int ba = blockIdx.x * blockDim.x + threadIdx.x;
    if (ba >= P * N) return;
    const int k = ba / N, i = ba - k * N;
    const int cid = cell_id[ba];
    const int slot = atomicAdd(cell_fill + (size_t)k * ncells + cid, 1);
    cell_tmp[(size_t)k * N + cell_start[(size_t)k * (ncells + 1) + cid] + slot] = i;
}

// Deterministic order inside every cell: rank each member by its atom index (one warp per cell).
__global__ void cell_sort_kernel(int P, int N, int ncells, const int* __restrict__ cell_start,
                                 const int* __restrict__ cell_tmp, const double* __restrict__ wtmp,
                                 const int* __restrict__ types, double4* __restrict__ wsorted) {
    const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= P * ncells) return;
    const int k = wid / ncells, c = wid - k * ncells;
    const int s0 = cell_start[(size_t)k * (ncells + 1) + c], s1 = cell_start[(size_t)k * (ncells + 1) + c + 1];
    const int* mem = cell_tmp + (size_t)k * N;
    for (int q = s0 + lane; q < s1; q += 32) {
        const int me = mem[q];
        int rank = 0;
        for (int t = s0; t < s1; ++t) rank += (mem[t] < me) ? 1 : 0;
        const size_t ba = (size_t)k * N + me;
        double4 o;
        o.x = wtmp[ba * 3]; o.y = wtmp[ba * 3 + 1]; o.z = wtmp[ba * 3 + 2];
        o.w = __longlong_as_double(((long long)types[me] << 32) | (long long)me);
        wsorted[(size_t)k * N + s0 + rank] = o;
    }
}

struct EnvConsts {
    double rc, rs, rc2, inv_range;   // inv_range = 1/(rc - rs)
    int ntypes;
    int sel[PIMD_MAX_TYPES];
    int seloff[PIMD_MAX_TYPES + 1];
    int nsel;
};

// One warp per centre bead-atom.
__global__ void __launch_bounds__(128)
neighbor_env_kernel(int P, int N, GridGeom g, EnvConsts ec, const double* __restrict__ wtmp,
                    const int* __restrict__ cell_id, const int* __restrict__ cell_start,
                    const double4* __restrict__ wsorted, int* __restrict__ ncount, NeighSlotA* __restrict__ slotA,
                    NeighSlotB* __restrict__ slotB, int* __restrict__ overflow) {
    const int ba = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (ba >= P * N) return;
    const int k = ba / N, i = ba - k * N;
    double gL[3], ginv_w[3], gcw[3];
    load_geom(g, gL, ginv_w);
    load_widths(g, gL, gcw);
    const double wi[3] = {wtmp[(size_t)ba * 3], wtmp[(size_t)ba * 3 + 1], wtmp[(size_t)ba * 3 + 2]};
    const int cid = cell_id[ba];
    const int c0 = cid % g.nc[0], c1 = (cid / g.nc[0]) % g.nc[1], c2 = cid / (g.nc[0] * g.nc[1]);
    const int* cs = cell_start + (size_t)k * (g.ncells + 1);
    const double4* ws = wsorted + (size_t)k * N;
    int cnt[PIMD_MAX_TYPES];
#pragma unroll
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) cnt[t] = 0;
    const unsigned lt_mask = (1u << lane) - 1u;
    const size_t slot0 = (size_t)ba * ec.nsel;

    // The (2R+1)^3 neighbour cells are taken in the order (oz, oy, ox), ox fastest.  Lane l of a batch looks up
    // cell l's range and periodic image first (27 independent loads instead of 27 dependent ones); the candidates
    // of all cells of the batch are then walked as one flat list, 32 at a time.
    const int nx_c = 2 * g.R[0] + 1, ny_c = 2 * g.R[1] + 1, nz_c = 2 * g.R[2] + 1;
    const int ncl = nx_c * ny_c * nz_c;
    const int mag_x = 65536 / nx_c + 1, mag_y = 65536 / ny_c + 1;     // exact for numerators < 343 and divisors <= 7
    for (int base = 0; base < ncl; base += 32) {
        int my_s0 = 0, my_s1 = 0, my_code = 0;
        {
            const int idx = base + lane;
            if (idx < ncl) {
                // idx -> (ox, oy, oz) and the periodic image of each coordinate without integer divisions: idx < 343
                // (R <= 3), so a 16-bit reciprocal is exact; |offset| <= R <= 3 cells, so the image is found by at
                // most three conditional steps per side (nc may be 1: configs[0])
                const int t1 = (idx * mag_x) >> 16;                 // idx / nx_c
                const int t2 = (t1 * mag_y) >> 16;                  // idx / (nx_c ny_c)
                const int ox = idx - t1 * nx_c - g.R[0], oy = t1 - t2 * ny_c - g.R[1], oz = t2 - g.R[2];
                const int xx = c0 + ox, yy = c1 + oy, zz = c2 + oz;
                int wx = xx, wy = yy, wz = zz, nx = 0, ny = 0, nz = 0;
#pragma unroll
                for (int it = 0; it < 3; ++it) {
                    if (wx < 0) { wx += g.nc[0]; --nx; } else if (wx >= g.nc[0]) { wx -= g.nc[0]; ++nx; }
                    if (wy < 0) { wy += g.nc[1]; --ny; } else if (wy >= g.nc[1]) { wy -= g.nc[1]; ++ny; }
                    if (wz < 0) { wz += g.nc[2]; --nz; } else if (wz >= g.nc[2]) { wz -= g.nc[2]; ++nz; }
                }
                const int cc = (wz * g.nc[1] + wy) * g.nc[0] + wx;
                my_s0 = cs[cc]; my_s1 = cs[cc + 1];
                // prune cells that lie entirely outside the cutoff sphere (about a third of the 27): distance from
                // the centre to the cell's box in the unwrapped cell frame, with a 1e-6 relative margin on r^2 that
                // dwarfs the rounding of the binning, so no candidate the exact test would accept is dropped
                const int un[3] = {xx, yy, zz};
                double dm2 = 0.0;
#pragma unroll
                for (int ax = 0; ax < 3; ++ax) {
                    const double wc = gcw[ax];
                    const double lo = un[ax] * wc - wi[ax], hi = wi[ax] - (un[ax] + 1) * wc;
                    const double dd = fmax(fmax(lo, hi), 0.0);
                    dm2 += dd * dd;
                }
                if (dm2 > ec.rc2 * (1.0 + 1e-6)) my_s1 = my_s0;
                my_code = (nx + 3) | ((ny + 3) << 3) | ((nz + 3) << 6);
            }
        }
        // The candidates of the non-pruned cells form one flat list in the same (oz, oy, ox) / in-cell order; it is
        // walked 32 at a time with every lane busy (cells hold ~24 atoms, so a batch per cell left a quarter of the
        // lanes idle and paid a per-cell header).
        // non-empty cells compacted to the low lanes (their order kept), prefix sums of their lengths
        const unsigned ne = __ballot_sync(0xffffffffu, my_s1 > my_s0);
        const int nne = __popc(ne);
        const int srcl = (int)(__fns(ne, 0, lane + 1) & 31u);          // lane of the (lane+1)-th non-empty cell
        const int c_s0 = __shfl_sync(0xffffffffu, my_s0, srcl);
        const int c_code = __shfl_sync(0xffffffffu, my_code, srcl);
        int c_len = __shfl_sync(0xffffffffu, my_s1, srcl) - c_s0;
        if (lane >= nne) c_len = 0;
        int pre = c_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, pre, o);
            if (lane >= o) pre += t;
        }
        const int total = __shfl_sync(0xffffffffu, pre, 31);
        const int c_beg = pre - c_len;
        // Batches are located in order.  The cells that START inside the batch [g0, g0 + 32) are marked in a 32-bit
        // mask (one warp OR-reduction); candidate g0 + l then belongs to cell cprev + popc(mask bits 0..l), cprev
        // being the last cell started before the batch.
        int cprev = -1;
        auto locate = [&](int g0, int& q, int& code) {
            const int rel = c_beg - g0;
            const unsigned bit = (lane < nne && rel >= 0 && rel < 32) ? (1u << rel) : 0u;
            const unsigned heads = __reduce_or_sync(0xffffffffu, bit);
            const int c = min(cprev + __popc(heads & (0xffffffffu >> (31 - lane))), 31);
            cprev += __popc(heads);
            const int cbeg = __shfl_sync(0xffffffffu, c_beg, c), cs0 = __shfl_sync(0xffffffffu, c_s0, c);
            code = __shfl_sync(0xffffffffu, c_code, c);
            q = cs0 + (g0 + lane - cbeg);
        };
        int qn = 0, coden = 0;
        double4 wn = make_double4(0, 0, 0, 0);
        if (total > 0) {
            locate(0, qn, coden);
            if (lane < total) wn = ws[qn];
        }
        for (int g0 = 0; g0 < total; g0 += 32) {
            const int q = qn, code = coden;
            const double4 wj = wn;
            const bool act = g0 + lane < total;
            if (g0 + 32 < total) {                              // next batch in flight while this one is tested
                locate(g0 + 32, qn, coden);
                if (g0 + 32 + lane < total) wn = ws[qn];
            }
            const int nx = (code & 7) - 3, ny = ((code >> 3) & 7) - 3, nz = ((code >> 6) & 7) - 3;
            bool keep = false;
            int tj = 0, j = 0;
            if (act) {
                const double sh[3] = {__dmul_rn((double)nx, gL[0]), __dmul_rn((double)ny, gL[1]),
                                      __dmul_rn((double)nz, gL[2])};
                const long long pk = __double_as_longlong(wj.w);
                j = (int)(pk & 0xffffffffll);
                tj = (int)(pk >> 32);
                const double d0 = __dadd_rn(__dsub_rn(wj.x, wi[0]), sh[0]);
                const double d1 = __dadd_rn(__dsub_rn(wj.y, wi[1]), sh[1]);
                const double d2 = __dadd_rn(__dsub_rn(wj.z, wi[2]), sh[2]);
                const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d0, d0), __dmul_rn(d1, d1)), __dmul_rn(d2, d2));
                keep = (r2 < ec.rc2) && !(code == (3 | (3 << 3) | (3 << 6)) && j == i);
            }
            // slot inside the type partition
            int slot = -1, sel_t = 0, seloff_t = 0;
            if (ec.ntypes == 2) {
                // the water case: two ballots instead of one per possible type
                const unsigned mk_all = __ballot_sync(0xffffffffu, keep);
                const unsigned mk0 = __ballot_sync(0xffffffffu, keep && tj == 0);
                const unsigned mk1 = mk_all & ~mk0;
                if (keep) {
                    const bool t0 = tj == 0;
                    slot = t0 ? cnt[0] + __popc(mk0 & lt_mask) : cnt[1] + __popc(mk1 & lt_mask);
                    sel_t = t0 ? ec.sel[0] : ec.sel[1];
                    seloff_t = t0 ? ec.seloff[0] : ec.seloff[1];
                }
                cnt[0] += __popc(mk0);
                cnt[1] += __popc(mk1);
            } else {
#pragma unroll
                for (int t = 0; t < PIMD_MAX_TYPES; ++t) {
                    if (t < ec.ntypes) {
                        const bool mine = keep && tj == t;
                        const unsigned mk = __ballot_sync(0xffffffffu, mine);
                        if (mine) { slot = cnt[t] + __popc(mk & lt_mask); sel_t = ec.sel[t]; seloff_t = ec.seloff[t]; }
                        cnt[t] += __popc(mk);
                    }
                }
            }
            if (keep) {
                if (slot >= sel_t) {
                    atomicOr(overflow, 1);
                    atomicMin(reinterpret_cast<unsigned*>(overflow) + 1, (unsigned)overflow[2]);    // which evaluation
                } else {
                    // queue the accepted candidate in its final slot: {j | image code, index into the cell-sorted
                    // positions}.  The FP64 environment arithmetic runs afterwards over the compact slots with all
                    // lanes busy (inside this loop only ~20 % of the lanes would be active).
                    *reinterpret_cast<uint4*>(slotB + slot0 + seloff_t + slot) =
                        make_uint4(0u, 0u, (uint32_t)j | ((uint32_t)code << 23), (uint32_t)q);     // {ds, rinv, jcode, pad}
                }
            }
        }
    }
    __syncwarp();
    // environment rows in FP64 (R-12), stored FP32: same operation order as the distance test above, so d and r2
    // are reproduced bit for bit
#pragma unroll
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) {
        if (t >= ec.ntypes) continue;
        const int n = min(cnt[t], ec.sel[t]);
        for (int e = lane; e < n; e += 32) {
            const size_t o = slot0 + ec.seloff[t] + e;
            NeighSlotB B = slotB[o];
            const uint32_t code = B.jcode >> 23;
            const int nx = (int)(code & 7) - 3, ny = (int)((code >> 3) & 7) - 3, nz = (int)((code >> 6) & 7) - 3;
            const double4 wj = ws[__float_as_int(B.pad)];
            double d[3];
            d[0] = __dadd_rn(__dsub_rn(wj.x, wi[0]), __dmul_rn((double)nx, gL[0]));
            d[1] = __dadd_rn(__dsub_rn(wj.y, wi[1]), __dmul_rn((double)ny, gL[1]));
            d[2] = __dadd_rn(__dsub_rn(wj.z, wi[2]), __dmul_rn((double)nz, gL[2]));
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
            const double r = sqrt(r2);
            if (r < 0.01) {          // |R| = 1/r > 100: beyond what the fixed FP16 scales of the descriptor kernels hold
                atomicOr(overflow, 8);
                atomicMin(reinterpret_cast<unsigned*>(overflow) + 1, (unsigned)overflow[2]);
            }
            double sw = 1.0, dsw = 0.0;
            if (r >= ec.rs) {
                const double u = (r - ec.rs) * ec.inv_range;
                sw = u * u * u * (-6.0 * u * u + 15.0 * u - 10.0) + 1.0;
                dsw = -30.0 * u * u * (u - 1.0) * (u - 1.0) * ec.inv_range;
            }
            const double rinv = 1.0 / r;
            const double sv = sw * rinv;
            const double ds = dsw * rinv - sw * rinv * rinv;
            NeighSlotA A;
            A.dx = (float)d[0]; A.dy = (float)d[1]; A.dz = (float)d[2]; A.s = (float)sv;
            B.ds = (float)ds; B.rinv = (float)rinv; B.pad = 0.f;
            slotA[o] = A;
            slotB[o] = B;
        }
    }
    if (lane == 0) {
#pragma unroll
        for (int t = 0; t < PIMD_MAX_TYPES; ++t)
            if (t < ec.ntypes) ncount[(size_t)ba * ec.ntypes + t] = min(cnt[t], ec.sel[t]);
    }
}

int neighbor_build(Model& m, const ForceArgs& a, cudaStream_t s) {
    const int PN = a.P * a.N;
    GridGeom g;
    for (int c = 0; c < 3; ++c) {
        g.L[c] = a.box[c];
        g.nc[c] = m.ncell[c];
        g.R[c] = m.R[c];
        g.inv_w[c] = (double)m.ncell[c] / a.box[c];
        g.cw[c] = a.box[c] / (double)m.ncell[c];
        g.inv_nc[c] = 1.0 / (double)m.ncell[c];
    }
    g.ncells = m.ncells;
    g.boxp = a.box_dev; g.rc = m.d.rcut; g.overflow = m.overflow; g.ctl = a.ctl;
    EnvConsts ec;
    ec.rc = m.d.rcut; ec.rs = m.d.rcut_smth; ec.rc2 = m.d.rcut * m.d.rcut;
    ec.inv_range = 1.0 / (m.d.rcut - m.d.rcut_smth);
    ec.ntypes = a.ntypes; ec.nsel = m.nsel;
    for (int t = 0; t < PIMD_MAX_TYPES; ++t) { ec.sel[t] = t < a.ntypes ? m.d.sel[t] : 0; ec.seloff[t] = m.seloff[t]; }
    ec.seloff[PIMD_MAX_TYPES] = m.nsel;

    cudaMemsetAsync(m.cell_count, 0, sizeof(int) * (size_t)a.P * (m.ncells + 1), s);
    cudaMemsetAsync(m.cell_fill, 0, sizeof(int) * (size_t)a.P * m.ncells, s);
    const int th = 128;
    wrap_bin_kernel<<<(PN + th - 1) / th, th, 0, s>>>(a.P, a.N, g, a.x, m.wtmp, m.cell_id, m.cell_count);
    cell_scan_kernel<<<a.P, 256, 0, s>>>(m.ncells, m.cell_count, m.cell_start);
    cell_fill_kernel<<<(PN + th - 1) / th, th, 0, s>>>(a.P, a.N, m.ncells, m.cell_id, m.cell_start, m.cell_fill,
                                                       m.cell_tmp);
    const long long nw = (long long)a.P * m.ncells;
    cell_sort_kernel<<<(unsigned)((nw * 32 + th - 1) / th), th, 0, s>>>(a.P, a.N, m.ncells, m.cell_start, m.cell_tmp,
                                                                        m.wtmp, a.types, m.wsorted);
    neighbor_env_kernel<<<(unsigned)(((long long)PN * 32 + th - 1) / th), th, 0, s>>>(
        a.P, a.N, g, ec, m.wtmp, m.cell_id, m.cell_start, m.wsorted, m.ncount, m.slotA, m.slotB, m.overflow);
    return 5;
}

}  // namespace pimd
