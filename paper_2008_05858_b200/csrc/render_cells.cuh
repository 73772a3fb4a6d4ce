// render_cells.cuh -- the cell-moment render in two kernels (round 2).
//
// render_moment_kernel does everything for a cell in one warp: batch prologue (sample loads, footprint boxes, phase powers),
// step 1 (the cell's weighted phase moments M), steps 2 + 3 (the contraction with the pixel-phase tables) and the write-out.
// On sm_100a the scalar fp64 instructions of one warp's prologue STARVE while other warps of its scheduler stream DMMAs
// (e2e_probe_fp64_pipe: 0.0008 instead of 1.22 warp instructions per clock), so the prologues and the contraction do not
// overlap the way five warps per scheduler suggest.  Here the two halves run as two kernels:
//
//   cell_moment_kernel  prologue + step 1 for every cell of every item, in any order (a cell's moments depend on nothing but
//                       its own samples); writes per cell a 32-byte header (footprint box, y-phase window) and the moment
//                       tiles in DMMA fragment order (32 lanes x 2 NPT doubles: 1 KB for NPT = 2) to the workspace.
//                       COUNT = true: the same walk without arithmetic, counting the cells of each item (once per plan).
//   cell_flush_kernel   steps 2 + 3 + a5 for the cells of an item in order, under the ticket queue and dependency counters of
//                       render_moment.cuh: DMMAs, table loads and the frame reductions only -- no scalar fp64 at all.
//
// The cell walk (where a cell ends) and the arithmetic are those of render_moment_kernel, operation for operation, so the frame
// has the same bits as the one-kernel form's (which still renders analytic PSF maps).  The batch call (e2e_render_frames) runs
// these kernels with the frames interleaved in one grid (BATCH).
#pragma once
#include "common.cuh"
#include "render_moment.cuh"

namespace e2e {

constexpr int kCellWarps = 4;          // warps per CTA of cell_moment_kernel (one item per warp)

struct CellHeader {                    // 32 bytes
    int i0, i1, j0, j1;                // footprint box of the cell (G9)
    int yb;                            // y-phase window
    int pad[3];
};

// per-item cell ranges and the record arrays in the workspace
struct CellStore {
    const long long* cell_off;         // [n_items + 1] first cell of every item (from the counting pass of the plan)
    CellHeader* hdr;                   // [n_cells]
    double* mom;                       // [n_cells][32 lanes][2 NPT]
    long long frame_cells;             // batch render: the records of frame b start at cell b * frame_cells of both arrays
    int n_frames;                      // batch render: 1-D grid, frame = blockIdx.x % n_frames (the frames advance together: a
                                       // grid.y per frame would run them one after the other, each at its own serial chain)
};

// FUSED: steps a1-a3 run here (setup.cuh's device functions: the oracle's operation sequence, the same bits as
// setup_samples_kernel) and the samples are never materialised; else they are read from the arrays setup_samples_kernel wrote
// NPT = 2: 8 CTAs per SM (64 registers; the shared-memory staging allows 8), measured 1.41 against 1.43 ms at 7 CTAs
// BATCH (e2e_render_frames): frame = blockIdx.x % n_frames; same geometry, the frame's own spectra (sp_batch[frame], device
// memory) and record region
template <int NPT, bool COUNT, bool FUSED, bool BATCH = false>
__global__ void __launch_bounds__(kCellWarps * 32, NPT == 2 ? 8 : 0)
cell_moment_kernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ ws,
                   const Strip* __restrict__ strips, const Item* __restrict__ items, const int* __restrict__ ids, int n_items,
                   MomentParam Q, CellStore C, int* __restrict__ counts, const __grid_constant__ FormatView F,
                   const __grid_constant__ SpectraParam SP, double2* __restrict__ zero, long long n_zero,
                   const SpectraParam* __restrict__ sp_batch)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // zero-fill of the frame (accumulate = 0) rides along: this kernel leaves most of the HBM bandwidth unused and touches no
    // pixel, and the flush kernel starts after it in stream order.  n_zero 16-byte elements, grid-stride.
    if (!COUNT && zero)
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_zero; i += (long long)gridDim.x * blockDim.x)
            __stcs(zero + i, make_double2(0.0, 0.0));
    const int bframe = BATCH ? (int)(blockIdx.x % (unsigned)C.n_frames) : 0;
    const int slot = (BATCH ? (int)(blockIdx.x / (unsigned)C.n_frames) : (int)blockIdx.x) * kCellWarps + warp;
    if (slot >= n_items) return;
    const int item_id = ids ? ids[slot] : slot;              // ids: the items of one row band (host path), else all of them
    MomentWarpSmem<NPT, false>& S = reinterpret_cast<MomentWarpSmem<NPT, false>*>(smem_raw)[warp];
    const int lq = lane >> 2, lr = lane & 3;
    constexpr int NP = 8 * NPT;
    const double ywin = 1.0 / (double)Q.nyb;
    const Item it = items[item_id];
    const Strip st = strips[it.strip];
    long long k = (long long)it.chunk0 * 32;
    long long kend = k + (long long)it.nchunks * 32;
    if (kend > st.n) kend = st.n;

    double mt[NPT][2];
    bool have = false;
    int cI0 = 0, cI1 = 0, cJ0 = 0, cJ1 = 0, cYb = 0;
    double cYc = 0.0;
    long long cell = COUNT ? 0 : C.cell_off[item_id] + (BATCH ? (long long)bframe * C.frame_cells : 0);
    int n_cells = 0;

    // the open cell is complete: hand it to the flush kernel
    auto emit = [&]() {
        if (!COUNT) {
            if (lane == 0) {                                   // the header as two 16-byte stores
                int4* hd = reinterpret_cast<int4*>(C.hdr + cell);
                hd[0] = make_int4(cI0, cI1, cJ0, cJ1);
                hd[1] = make_int4(cYb, 0, 0, 0);
            }
            double* dst = C.mom + ((size_t)cell * 32 + lane) * (2 * NPT);
#pragma unroll
            for (int qt = 0; qt < NPT; ++qt) *reinterpret_cast<double2*>(dst + 2 * qt) = make_double2(mt[qt][0], mt[qt][1]);
            cell += 1;
        }
        n_cells += 1;
    };

    while (k < kend) {
        const int nb = (int)min((long long)32, kend - k);
        const bool valid = lane < nb;
        double xk, yk, wk = 0.0;
        if (COUNT || FUSED) {
            // positions straight from the format (a1, a3: the setup kernel's operations, so the cells are the render's)
            const int fiber = it.strip / F.n_orders, o = it.strip - fiber * F.n_orders;
            double lam, X, Y;
            sample_position_fast(F, o, k + (valid ? lane : nb - 1), lam, X, Y);
            xk = __dadd_rn(X, F.fiber_dx[fiber]);
            yk = __dadd_rn(Y, F.fiber_dy[fiber]);
            if (FUSED && !COUNT) {                              // a2: the photon weight, setup_samples_kernel's expression
                const e2e_spectrum_t& sf = BATCH ? sp_batch[bframe].s[fiber] : SP.s[fiber];
                const double wv = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(sf.scale, spectrum_at(sf, lam)), blaze_at(F, o, lam)),
                                                      eff_at(F, lam)), F.dl[o]);
                wk = valid ? wv : 0.0;
            }
        } else {
            const long long kidx = st.off + k + (valid ? lane : nb - 1);
            xk = __ldcs(xs + kidx); yk = __ldcs(ys + kidx);
            wk = valid ? __ldcs(ws + kidx) : 0.0;
        }
        // G9 footprint box (same operations as the oracle's box)
        const int ilo = __double2int_ru(__dsub_rn(xk, Q.hbx)), ihi = __double2int_rd(__dadd_rn(xk, Q.hbx));
        const int jlo = __double2int_ru(__dsub_rn(yk, Q.hby)), jhi = __double2int_rd(__dadd_rn(yk, Q.hby));
        const double dx = __dsub_rn(__dsub_rn(xk, (double)ilo), Q.c0x);
        const double dy = __dsub_rn(__dsub_rn(yk, (double)jlo), Q.c0y);
        if (!COUNT) {
            __syncwarp();                                      // previous batch's readers are done
            double v[NP];
            v[0] = wk;
            double sq = dx;
#pragma unroll
            for (int h = 1; h < NP; h *= 2) {
#pragma unroll
                for (int p = 0; p < h; ++p)
                    if (h + p < NP) v[h + p] = v[p] * sq;
                sq *= sq;
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) S.vx[p * kMomLdk + lane] = v[p];
            __syncwarp();
        }
        int pos = 0;
        while (pos < nb) {
            const int kI0 = __shfl_sync(0xffffffffu, ilo, pos), kI1 = __shfl_sync(0xffffffffu, ihi, pos);
            const int kJ0 = __shfl_sync(0xffffffffu, jlo, pos), kJ1 = __shfl_sync(0xffffffffu, jhi, pos);
            const double kdy = __shfl_sync(0xffffffffu, dy, pos);
            if (have && (kI0 != cI0 || kI1 != cI1 || kJ0 != cJ0 || kJ1 != cJ1 || !(fabs(kdy - cYc) <= ywin))) {
                emit();
                have = false;
            }
            if (!have) {
                have = true;
                cI0 = kI0; cI1 = kI1; cJ0 = kJ0; cJ1 = kJ1;
                cYb = min(max((int)floor((kdy + 0.5) * (double)Q.nyb), 0), Q.nyb - 1);
                cYc = ((double)cYb + 0.5) * ywin - 0.5;
#pragma unroll
                for (int a = 0; a < NPT; ++a) { mt[a][0] = 0.0; mt[a][1] = 0.0; }
            }
            const double dl = dy - cYc;
            const unsigned same = __ballot_sync(0xffffffffu, valid && ilo == cI0 && ihi == cI1 && jlo == cJ0 && jhi == cJ1 &&
                                                                 fabs(dl) <= ywin);
            const unsigned rest = ~(same >> pos);
            const int run = rest ? (__ffs(rest) - 1) : 32;
            const int pend = min(pos + run, nb);
            if (!COUNT) {
                __syncwarp();                                  // the previous run's step-1 reads of vy are done
                // samples outside the run [pos, pend) stage zeros: the k-steps at the run's ends need no select
                const bool mine = lane >= pos && lane < pend;
                const double d1 = mine ? dl : 0.0;
                const double d2 = d1 * d1, d3 = d2 * d1, d4 = d2 * d2;
                S.vy[0 * kMomLdk + lane] = mine ? 1.0 : 0.0;
                S.vy[1 * kMomLdk + lane] = d1;
                S.vy[2 * kMomLdk + lane] = d2;
                S.vy[3 * kMomLdk + lane] = d3;
                S.vy[4 * kMomLdk + lane] = d4;
                S.vy[5 * kMomLdk + lane] = d4 * d1;
                S.vy[6 * kMomLdk + lane] = d4 * d2;
                S.vy[7 * kMomLdk + lane] = d4 * d3;
                __syncwarp();
                // ---- step 1: MT += VX VY^T over the samples [pos, pend)
                for (int ks = pos >> 2; ks <= (pend - 1) >> 2; ++ks) {
                    const int ksamp = 4 * ks + lr;
                    const double a = S.vy[lq * kMomLdk + ksamp];
                    double b[NPT];
#pragma unroll
                    for (int qt = 0; qt < NPT; ++qt) b[qt] = S.vx[(8 * qt + lq) * kMomLdk + ksamp];
#pragma unroll
                    for (int qt = 0; qt < NPT; ++qt) dmma_m8n8k4(mt[qt][0], mt[qt][1], a, b[qt]);
                }
            }
            pos = pend;
        }
        k += nb;
    }
    if (have) emit();
    if (COUNT && lane == 0) counts[item_id] = n_cells;
}

// steps 2 + 3 + a5 for the cells of one item, in order, under the ticket queue (render_moment.cuh queue_take / queue_done)
// BATCH (e2e_render_frames): frame = blockIdx.x % n_frames, with its own target, control block and record region
template <int NPT, bool BATCH = false>
__global__ void __launch_bounds__(32, NPT == 2 ? E2E_MOM_MINB : 1)
cell_flush_kernel(QueueParam W, MomentParam Q, CellStore C, double* __restrict__ frame, int nx, int ny, double* const* __restrict__ frames)
{
    const int lane = threadIdx.x & 31;
    unsigned* ctrl = W.ctrl;
    long long cbase = 0;
    if (BATCH) {
        const unsigned b = blockIdx.x % (unsigned)C.n_frames;
        frame = frames[b];
        ctrl += (long long)b * W.ctrl_stride;
        cbase = (long long)b * C.frame_cells;
    }
    const int item_id = queue_take(W, ctrl, lane);
    if (item_id < 0) return;
    const long long c0 = C.cell_off[item_id] + cbase, c1 = C.cell_off[item_id + 1] + cbase;
    for (long long cell = c0; cell < c1; ++cell) {
        const CellHeader h = C.hdr[cell];
        double mt[1][NPT][2];
        const double* src = C.mom + ((size_t)cell * 32 + lane) * (2 * NPT);
#pragma unroll
        for (int qt = 0; qt < NPT; ++qt) {
            const double2 v = __ldcs(reinterpret_cast<const double2*>(src + 2 * qt));
            mt[0][qt][0] = v.x; mt[0][qt][1] = v.y;
        }
        moment_flush_cell<NPT, false>(Q, mt, h.i0, h.i1, h.j0, h.j1, h.yb, 0, 0, frame, nx, ny, lane);
    }
    queue_done(W, ctrl, item_id, lane);
}

// ---- small frames (a single strip, a few hundred items): the launch cannot fill the GPU, the frame time is the serial chain of
// cells that share pixels, and one warp per cell (180 dependent-ish DMMAs, ~4 us) is the wrong shape.  Here one CTA of kWideWarps
// warps renders an item: every warp owns 8 x 8 tiles of the window (tile w, w + kWideWarps, ...), computes Y_t for its column tile
// itself (redundantly across the row tiles) and contracts it with its row tile's cy: (2 NPT + 2) T DMMAs per tile and cell
// instead of 30 T in one warp.  Every output element sees the same DMMA sequence as in moment_flush_cell (terms in order, k-slot x
// then y; Y_t by power tile, x then y): the frame has the same bits.  Consecutive cells of the item overlap, and their tiles
// belong to different warps, so a CTA barrier (instead of __syncwarp) orders one cell's reductions before the next cell's.
constexpr int kWideWarps = 9;
template <int NPT, bool BATCH = false>
__global__ void __launch_bounds__(kWideWarps * 32)
cell_flush_wide_kernel(QueueParam W, MomentParam Q, CellStore C, double* __restrict__ frame, int nx, int ny,
                       double* const* __restrict__ frames)
{
    __shared__ int s_item;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lq = lane >> 2, lr = lane & 3;
    unsigned* ctrl = W.ctrl;
    long long cbase = 0;
    if (BATCH) {                                               // e2e_render_frames
        const unsigned b = blockIdx.x % (unsigned)C.n_frames;
        frame = frames[b];
        ctrl += (long long)b * W.ctrl_stride;
        cbase = (long long)b * C.frame_cells;
    }
    if (warp == 0) {
        const int id = queue_ticket(W, ctrl, lane);
        if (lane == 0) s_item = id;
    }
    __syncthreads();
    const int item_id = s_item;
    if (item_id < 0) return;
    const long long c0 = C.cell_off[item_id] + cbase, c1 = C.cell_off[item_id + 1] + cbase;
    // the first record travels while warp 0 waits for the item's dependencies (records are final before this launch)
    CellHeader hn = {};
    double2 mn[NPT] = {};
    auto fetch = [&](long long cell) {
        hn = C.hdr[cell];
        const double* src = C.mom + ((size_t)cell * 32 + lane) * (2 * NPT);
#pragma unroll
        for (int qt = 0; qt < NPT; ++qt) mn[qt] = __ldg(reinterpret_cast<const double2*>(src + 2 * qt));
    };
    if (c0 < c1) fetch(c0);
    if (warp == 0) queue_wait(ctrl, item_id);
    __syncthreads();
    const int ntile = Q.nit * Q.njt;
    for (long long cell = c0; cell < c1; ++cell) {
        const CellHeader h = hn;
        double mc[NPT][2];
#pragma unroll
        for (int qt = 0; qt < NPT; ++qt) { mc[qt][0] = mn[qt].x; mc[qt][1] = mn[qt].y; }
        if (cell + 1 < c1) fetch(cell + 1);
        const bool dead = h.i1 < 0 || h.i0 >= nx || h.j1 < 0 || h.j0 >= ny || h.i1 < h.i0 || h.j1 < h.j0;
        const int rlim = min(h.j1, ny - 1), clim = min(h.i1, nx - 1);
        for (int tile = warp; tile < ntile && !dead; tile += kWideWarps) {
            const int it = tile / Q.njt, jt = tile - it * Q.njt;
            if (h.i0 + 8 * it > clim || h.j0 + 8 * jt > rlim) continue;
            double o0 = 0.0, o1 = 0.0;
#pragma unroll 2
            for (int t = 0; t < Q.T; ++t) {
                const double2 cy = __ldg(Q.fy + ((size_t)(h.yb * Q.T + t) * Q.njt + jt) * 32 + lane);
                const double2* fx = Q.fx + ((size_t)(t * Q.nit + it) * NPT) * 32 + lane;
                double2 cx[NPT];
#pragma unroll
                for (int qt = 0; qt < NPT; ++qt) cx[qt] = __ldg(fx + qt * 32);
                double y0 = 0.0, y1 = 0.0;
#pragma unroll
                for (int qt = 0; qt < NPT; ++qt) {
                    dmma_m8n8k4(y0, y1, cx[qt].x, mc[qt][0]);
                    dmma_m8n8k4(y0, y1, cx[qt].y, mc[qt][1]);
                }
                dmma_m8n8k4(o0, o1, y0, cy.x);
                dmma_m8n8k4(o0, o1, y1, cy.y);
            }
            const int col = h.i0 + 8 * it + lq;
            const int row = h.j0 + 8 * jt + 2 * lr;
            if (col >= 0 && col <= clim) {
                if (row >= 0 && row <= rlim) atomicAdd(frame + (size_t)row * nx + col, o0);
                if (row + 1 >= 0 && row + 1 <= rlim) atomicAdd(frame + (size_t)(row + 1) * nx + col, o1);
            }
        }
        __syncthreads();                                       // the next cell's window overlaps this one
    }
    // every warp's reductions are performed before any successor's counter moves
    __threadfence();
    __syncthreads();
    if (warp == 0) {
        unsigned* const pend = ctrl + kCtrlHeads;
        const int s1 = W.succ_off[item_id + 1];
        for (int d = W.succ_off[item_id] + lane; d < s1; d += 32) red_release_dec_u32(pend + W.succ_idx[d]);
    }
}

}  // namespace e2e
