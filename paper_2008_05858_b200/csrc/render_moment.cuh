// render_moment.cuh -- steps a4 + a5 for the analytic PSF under dense sampling: the production kernel.
//
// A *cell* is a maximal run of consecutive samples of one strip that share one footprint box (G9):
// ilo = ceil(x - hbx), ihi = floor(x + hbx), jlo, jhi.  Inside a cell the pixel-integrated factors of chord term t
// are polynomials of the sample's phase (dx, dy) = ((x - ilo) - c0x, (y - jlo) - c0y) in (-1/2, 1/2]^2
// (poly_tables.h, truncation error < 1e-17):
//
//     AX_t[k][i] = sum_q cx_t[q][i] dx_k^q          BY_t[k][j] = sum_p cy_t[p][j] dy_k^p
//
// so the cell's whole contribution to the frame ("the sum of the single fibers image ... at each wavelength",
// P:79 "surface integral of the convolution ...") regroups exactly into
//
//     out[j][i] = sum_k w_k sum_t BY_t[k][j] AX_t[k][i] = sum_t ( cy_t^T  M  cx_t )[j][i],
//     M[p][q]   = sum_k w_k dy_k^p dx_k^q                                   (the cell's weighted phase moments)
//
// Per sample only the moment update is left; the cost per cell does not depend on how many samples the cell holds.
// The y-phase of one cell's samples moves by (trace slope) x (1 px) only, so BY uses one of nyb overlapping phase
// windows with its own degree-7 fit (poly_tables.h): p runs over 8 powers of delta = dy - (window centre) = ONE power
// tile, while q runs over the P + 1 powers of dx (the x-phase sweeps the whole pixel inside a cell).  A cell = maximal
// run of samples with one footprint box whose dy stays inside the window chosen at its first sample.
//
// Everything is a small dense fp64 contraction and runs as chained mma.sync.m8n8k4.f64 tiles (DMMA: same FP64 pipe as
// DFMA, 256 FMAs per instruction).  The products are ordered so that the short dimension (8 powers of delta) is the
// contraction index of the LARGE product, and transposed so that every C fragment feeds the next product's A operand
// directly from registers: lane l of a C tile holds columns 2(l%4)+{0,1}, and the k-slot l%4 of the next product is
// *defined* to be that column, with the table operand stored in the same permuted order:
//
//   step 1  M[p][q]      = sum_k dy_k^p (w_k dx_k^q)          A = VY (smem),      B = VX (smem)    C -> mt   NPT DMMAs / 4 samples
//   step 2  Y_t^T[i][p]  = sum_q cx_t[q][i] M[p][q]           A = fx table,       B = mt (regs)    C -> yt   ncol/8 * 2 NPT DMMAs
//   step 3  out^T[i][j] += sum_p Y_t^T[i][p] cy_t[p][j]       A = yt (regs),      B = fy table     C -> out  ncol/8 * nrow/8 * 2 DMMAs
//
// ESPRESSO-like PSF (24 x 24 window, T = 6, NPT = 2): 30 DMMAs per term, 180 per cell (the first version of this kernel,
// with both phases on the full range and the contraction over q last, needed 360).
//
// One warp per work item (run of consecutive 32-sample chunks of one strip) and per CTA, no block-level cooperation.  ONE
// launch renders a whole frame (or one row band of the host path): every warp takes the next item of the queue
// (atomic ticket), waits until the items it shares pixels with and that come earlier in the queue are done (its counter
// of unfinished dependencies reaches 0; the lists are built on the host, api.cu build_plan), renders, and decrements the
// counters of its successors.  A pixel's
// additions therefore happen in queue order whatever the timing -> bit-reproducible; inside a warp the finished windows
// are added to the frame by L2 reductions (red.global.add.f64) that the flush's __syncwarp() keeps in cell order.
// Deadlock-free: an item only waits for items taken before it, and a taken item is held by a running warp.
#pragma once
#include "common.cuh"
#include "render_poly.cuh"

namespace e2e {

#ifndef E2E_MOM_MINB
#define E2E_MOM_MINB 18          // single-warp CTAs per SM asked of ptxas for NPT = 2: 96 registers, no spills, 21 resident
                                 // (16 -> 114 registers: 6.13 ms; 17-19 -> 96: 6.00; 22-24 -> 80 with spills: 6.38)
#endif
constexpr int kMomWarps = 1;           // warps per CTA: one item per CTA, so a slow item never holds three finished warps' resources
                                       // (4 / 2 / 1 warps per CTA: 6.18 / 6.17 / 6.13 ms)
constexpr int kMomLdk = 36;            // pitch of the power arrays V[power][sample] (36 mod 16 = 4: conflict-free fragments)

template <int NPT, bool MAP = false>
struct MomentWarpSmem {
    double vx[8 * NPT * kMomLdk];      // w_k dx_k^q
    double vy[8 * kMomLdk];            // delta_k^p, p = 0..7 (rewritten for every cell: delta is relative to the cell's window)
    double beta[MAP ? 4 * kMomLdk : 1];// PSF map (G21): bilinear weight of each of the cell's 4 nodes at every sample
};

// work queue of one render launch
struct QueueParam {
    const int* queue;              // item ids in queue order, or nullptr (= 0 .. n - 1)
    int n;                         // items in the queue
    const int* succ_off;           // [n_items + 1] CSR: the items that wait for item i (its successors; ids > i)
    const int* succ_idx;
    const int* dep_off;            // [n_items + 1] CSR of the transposed lists (the items i waits for); e2e_plan_check only
    const int* dep_idx;
    unsigned* ctrl;                // control block, initialised before the launch: head counters, then per item the number
                                   // of its dependencies that are not finished yet
    int head;                      // which head counter this launch uses
    long long ctrl_stride;         // batch render: control block of frame b at ctrl + b * ctrl_stride (in unsigned)
};
constexpr int kCtrlHeads = 64;     // unsigned words before the counters

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_dec_u32(unsigned* p)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(0xffffffffu) : "memory");
}

// Take the next item of the queue and wait until its dependencies are finished.  The warp takes a TICKET rather than its
// block index: tickets are handed out in the order in which warps really start, so every item before this one in the queue
// is held by a warp that is already running (deadlock freedom).  The wait is a warp-uniform spin on ONE word (a per-lane
// loop over dependency flags made ptxas spill 500 bytes of the render loop's state at 96 registers).  Returns -1 when the
// queue is exhausted.
// ticket: the next item of the queue (-1: none left); the item may not touch the frame before queue_wait returns
__device__ __forceinline__ int queue_ticket(const QueueParam& W, unsigned* ctrl, int lane)
{
    unsigned qpos = 0;
    if (lane == 0) qpos = atomicAdd(ctrl + W.head, 1u);
    qpos = __shfl_sync(0xffffffffu, qpos, 0);
    if (qpos >= (unsigned)W.n) return -1;
    return W.queue ? W.queue[qpos] : (int)qpos;
}
__device__ __forceinline__ void queue_wait(unsigned* ctrl, int item_id)
{
    const unsigned* f = ctrl + kCtrlHeads + item_id;
    while (ld_acquire_u32(f) != 0u) __nanosleep(100);
    __syncwarp();
}
__device__ __forceinline__ int queue_take(const QueueParam& W, unsigned* ctrl, int lane)
{
    const int item_id = queue_ticket(W, ctrl, lane);
    if (item_id >= 0) queue_wait(ctrl, item_id);
    return item_id;
}

// Publish item_id as finished: every lane's frame reductions are performed (fence) before any successor's counter moves
// (warp barrier, then release reductions on the counters)
__device__ __forceinline__ void queue_done(const QueueParam& W, unsigned* ctrl, int item_id, int lane)
{
    __threadfence();
    __syncwarp();
    unsigned* const pend = ctrl + kCtrlHeads;
    const int s1 = W.succ_off[item_id + 1];
    for (int d = W.succ_off[item_id] + lane; d < s1; d += 32) red_release_dec_u32(pend + W.succ_idx[d]);
}

// steps 2 + 3 + a5 for one cell: its moment set(s) mt, footprint box, y-phase window and (MAP) node cell
template <int NPT, bool MAP>
__device__ __forceinline__ void moment_flush_cell(const MomentParam& Q, const double (&mt)[MAP ? 4 : 1][NPT][2], int cI0, int cI1, int cJ0,
                                                  int cJ1, int cYb, int cG, int cH, double* __restrict__ frame, int nx, int ny, int lane)
{
    constexpr int NC = MAP ? 4 : 1;
    const int lq = lane >> 2, lr = lane & 3;
    (void)cG; (void)cH;

        const bool dead = cI1 < 0 || cI0 >= nx || cJ1 < 0 || cJ0 >= ny || cI1 < cI0 || cJ1 < cJ0;
        if (dead) return;
        for (int jp = 0; jp < Q.njt; jp += 3) {
            if (cJ0 + 8 * jp > cJ1 || cJ0 + 8 * jp >= ny) break;
            for (int ip = 0; ip < Q.nit; ip += 3) {
                if (cI0 + 8 * ip > cI1 || cI0 + 8 * ip >= nx) break;
                double out[3][3][2];                           // [it][jt]: lane owns col 8 it + l/4, rows 8 jt + 2 (l%4) + {0,1}
#pragma unroll
                for (int a = 0; a < 3; ++a)
#pragma unroll
                    for (int b = 0; b < 3; ++b) { out[a][b][0] = 0.0; out[a][b][1] = 0.0; }
#pragma unroll 1
              for (int c = 0; c < NC; ++c) {
                size_t node = 0;
                if (MAP) {                                     // node c = 2 (row) + (column) of the cell's 4; absent on 1-wide grids
                    if (((c & 1) && Q.gx == 1) || ((c & 2) && Q.gy == 1)) continue;
                    node = (size_t)(cH + (c >> 1)) * Q.gx + (cG + (c & 1));
                }
                double mc[NPT][2];                             // this node's moment set (static register indices only)
#pragma unroll
                for (int cc = 0; cc < NC; ++cc)
                    if (cc == c) {
#pragma unroll
                        for (int qt = 0; qt < NPT; ++qt) { mc[qt][0] = mt[cc][qt][0]; mc[qt][1] = mt[cc][qt][1]; }
                    }
#pragma unroll 2                                        // two terms in flight: step 2 of one overlaps step 3 of the other
                for (int t = 0; t < Q.T; ++t) {
                    const double2* fy = Q.fy + node * Q.fy_node_stride + ((size_t)(cYb * Q.T + t) * Q.njt + jp) * 32 + lane;
                    const double2* fx = Q.fx + node * Q.fx_node_stride + ((size_t)(t * Q.nit + ip) * NPT) * 32 + lane;
                    double2 cy[3], cx[3][NPT];
#pragma unroll
                    for (int jt = 0; jt < 3; ++jt) cy[jt] = (jp + jt < Q.njt) ? __ldg(fy + jt * 32) : make_double2(0.0, 0.0);
#pragma unroll
                    for (int it = 0; it < 3; ++it)
#pragma unroll
                        for (int qt = 0; qt < NPT; ++qt)
                            cx[it][qt] = (ip + it < Q.nit) ? __ldg(fx + (it * NPT + qt) * 32) : make_double2(0.0, 0.0);
                    // ---- step 2: Y_t^T = cx_t^T M^T  (columns x 8 powers of delta; contraction over the powers of dx)
                    double yt[3][2];
#pragma unroll
                    for (int it = 0; it < 3; ++it) { yt[it][0] = 0.0; yt[it][1] = 0.0; }
#pragma unroll
                    for (int qt = 0; qt < NPT; ++qt) {
#pragma unroll
                        for (int it = 0; it < 3; ++it) dmma_m8n8k4(yt[it][0], yt[it][1], cx[it][qt].x, mc[qt][0]);
#pragma unroll
                        for (int it = 0; it < 3; ++it) dmma_m8n8k4(yt[it][0], yt[it][1], cx[it][qt].y, mc[qt][1]);
                    }
                    // ---- step 3: out^T += Y_t^T cy_t  (contraction over the 8 powers of delta: two k-slots)
#pragma unroll
                    for (int it = 0; it < 3; ++it)
#pragma unroll
                        for (int jt = 0; jt < 3; ++jt) dmma_m8n8k4(out[it][jt][0], out[it][jt][1], yt[it][0], cy[jt].x);
#pragma unroll
                    for (int it = 0; it < 3; ++it)
#pragma unroll
                        for (int jt = 0; jt < 3; ++jt) dmma_m8n8k4(out[it][jt][0], out[it][jt][1], yt[it][1], cy[jt].y);
                }
              }
                // ---- a5: add the panel to the frame by L2 reductions (red.global.add.f64): the same IEEE sum as load + add +
                // store without a round trip to wait for.  Order per pixel: items of one launch never share a pixel, and
                // inside the warp the __syncwarp() that closes every flush orders this cell's reductions before the next
                // cell's -> bit-reproducible
                const int rlim = min(cJ1, ny - 1), clim = min(cI1, nx - 1);
#pragma unroll
                for (int it = 0; it < 3; ++it) {
                    const int col = cI0 + 8 * (ip + it) + lq;
                    const bool cok = col >= 0 && col <= clim;
#pragma unroll
                    for (int jt = 0; jt < 3; ++jt)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int row = cJ0 + 8 * (jp + jt) + 2 * lr + e;
                            if (cok && row >= 0 && row <= rlim) atomicAdd(frame + (size_t)row * nx + col, out[it][jt][e]);
                        }
                }
            }
        }
        __syncwarp();                                          // the next cell's window overlaps this one
    }

// MAP (G21, analytic PSF map): the PSF of a sample is the bilinear blend of 4 node PSFs, and the blend is linear, so
// a cell (now also: one node cell of the map) keeps ONE weighted moment set per node, M_c = sum_k (w_k beta_c,k) delta^p dx^q, and
// its contribution is sum_c cy_c^T M_c cx_c with node c's own tables -- steps 2 + 3 run once per node into the same window.
template <int NPT, bool MAP>
__global__ void __launch_bounds__(kMomWarps * 32, MAP ? 12 : (NPT == 2 ? E2E_MOM_MINB : 1))
render_moment_kernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ ws,
                     const Strip* __restrict__ strips, const Item* __restrict__ items, QueueParam W, MomentParam Q,
                     double* __restrict__ frame, int nx, int ny, long long w_stride, double* const* __restrict__ frames)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (frames) {                                             // batch render (e2e_render_frames): blockIdx.y = frame,
        frame = frames[blockIdx.y];                           // same geometry, its own weights, target and control block
        ws += (long long)blockIdx.y * w_stride;
    }
    MomentWarpSmem<NPT, MAP>& S = reinterpret_cast<MomentWarpSmem<NPT, MAP>*>(smem_raw)[warp];
    constexpr int NC = MAP ? 4 : 1;                           // moment sets per cell
    const int lq = lane >> 2, lr = lane & 3;                  // fragment coordinates: l/4 and l%4
    constexpr int NP = 8 * NPT;
    const double ywin = 1.0 / (double)Q.nyb;

    const int item_id = queue_take(W, W.ctrl + (frames ? (long long)blockIdx.y * W.ctrl_stride : 0), lane);
    if (item_id < 0) return;
    const Item it = items[item_id];
    const Strip st = strips[it.strip];

    long long k = (long long)it.chunk0 * 32;
    long long kend = k + (long long)it.nchunks * 32;
    if (kend > st.n) kend = st.n;

    double mt[NC][NPT][2];                                     // M tiles [node][qt]: lane holds M[p = l/4][q = 8qt + 2(l%4) + e]
    bool have = false;
    int cI0 = 0, cI1 = 0, cJ0 = 0, cJ1 = 0, cYb = 0;           // footprint box and y-phase window of the open cell
    int cG = 0, cH = 0;                                        // MAP: its node cell (first node column / row)
    double cYc = 0.0;                                          // its centre

    // steps 2 + 3 + a5 for the open cell
    auto flush = [&]() { moment_flush_cell<NPT, MAP>(Q, mt, cI0, cI1, cJ0, cJ1, cYb, cG, cH, frame, nx, ny, lane); };

    while (k < kend) {
        // ---- next batch of up to 32 samples: footprint boxes, phases, power arrays
        const int nb = (int)min((long long)32, kend - k);
        const bool valid = lane < nb;
        const long long kidx = st.off + k + (valid ? lane : nb - 1);
        // streamed once: evict-first loads keep the L1 for the tables
        const double xk = __ldcs(xs + kidx), yk = __ldcs(ys + kidx);
        const double wk = valid ? __ldcs(ws + kidx) : 0.0;
        // G9 footprint box (same operations as the oracle's box)
        const int ilo = __double2int_ru(__dsub_rn(xk, Q.hbx)), ihi = __double2int_rd(__dadd_rn(xk, Q.hbx));
        const int jlo = __double2int_ru(__dsub_rn(yk, Q.hby)), jhi = __double2int_rd(__dadd_rn(yk, Q.hby));
        const double dx = __dsub_rn(__dsub_rn(xk, (double)ilo), Q.c0x);
        const double dy = __dsub_rn(__dsub_rn(yk, (double)jlo), Q.c0y);
        // MAP: node cell and bilinear weights of the sample (T3's rule: nodes at g (nx-1)/(gx-1), clamped outside the grid)
        int g0 = 0, h0 = 0;
        double bfx = 0.0, bfy = 0.0;
        if (MAP) {
            if (Q.gx > 1) {
                const double t = fmin(fmax(xk * Q.fsx, 0.0), (double)(Q.gx - 1));
                g0 = min((int)floor(t), Q.gx - 2);
                bfx = t - (double)g0;
            }
            if (Q.gy > 1) {
                const double t = fmin(fmax(yk * Q.fsy, 0.0), (double)(Q.gy - 1));
                h0 = min((int)floor(t), Q.gy - 2);
                bfy = t - (double)h0;
            }
        }
        __syncwarp();                                          // previous batch's readers are done
        if (MAP) {
            S.beta[0 * kMomLdk + lane] = (1.0 - bfy) * (1.0 - bfx);
            S.beta[1 * kMomLdk + lane] = (1.0 - bfy) * bfx;
            S.beta[2 * kMomLdk + lane] = bfy * (1.0 - bfx);
            S.beta[3 * kMomLdk + lane] = bfy * bfx;
        }
        {
            // w dx^p by repeated squaring: the same number of multiplications, dependency depth log2(NP) instead of NP
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
        }
        __syncwarp();
        int pos = 0;
        while (pos < nb) {
            const int kI0 = __shfl_sync(0xffffffffu, ilo, pos), kI1 = __shfl_sync(0xffffffffu, ihi, pos);
            const int kJ0 = __shfl_sync(0xffffffffu, jlo, pos), kJ1 = __shfl_sync(0xffffffffu, jhi, pos);
            const double kdy = __shfl_sync(0xffffffffu, dy, pos);
            const int kG = MAP ? __shfl_sync(0xffffffffu, g0, pos) : 0, kH = MAP ? __shfl_sync(0xffffffffu, h0, pos) : 0;
            if (have && (kI0 != cI0 || kI1 != cI1 || kJ0 != cJ0 || kJ1 != cJ1 || !(fabs(kdy - cYc) <= ywin) || kG != cG || kH != cH)) {
                flush();
                have = false;
            }
            if (!have) {
                have = true;
                cI0 = kI0; cI1 = kI1; cJ0 = kJ0; cJ1 = kJ1; cG = kG; cH = kH;
                // window whose centre is nearest to the first sample: |delta| <= ywin / 2, kept while |delta| <= ywin
                cYb = min(max((int)floor((kdy + 0.5) * (double)Q.nyb), 0), Q.nyb - 1);
                cYc = ((double)cYb + 0.5) * ywin - 0.5;
#pragma unroll
                for (int c = 0; c < NC; ++c)
#pragma unroll
                    for (int a = 0; a < NPT; ++a) { mt[c][a][0] = 0.0; mt[c][a][1] = 0.0; }
            }
            const double dl = dy - cYc;
            const unsigned same = __ballot_sync(0xffffffffu, valid && ilo == cI0 && ihi == cI1 && jlo == cJ0 && jhi == cJ1 &&
                                                                 fabs(dl) <= ywin && g0 == cG && h0 == cH);
            const unsigned rest = ~(same >> pos);              // bit r: sample pos + r is NOT in the cell
            const int run = rest ? (__ffs(rest) - 1) : 32;     // >= 1: sample pos is in
            const int pend = min(pos + run, nb);
            // powers of delta for this run (delta is relative to the cell's window, so they are staged per run)
            __syncwarp();                                      // the previous run's step-1 reads of vy are done
            {
                const double d2 = dl * dl, d3 = d2 * dl, d4 = d2 * d2;
                S.vy[0 * kMomLdk + lane] = 1.0;
                S.vy[1 * kMomLdk + lane] = dl;
                S.vy[2 * kMomLdk + lane] = d2;
                S.vy[3 * kMomLdk + lane] = d3;
                S.vy[4 * kMomLdk + lane] = d4;
                S.vy[5 * kMomLdk + lane] = d4 * dl;
                S.vy[6 * kMomLdk + lane] = d4 * d2;
                S.vy[7 * kMomLdk + lane] = d4 * d3;
            }
            __syncwarp();
            // ---- step 1: MT += VX VY^T over the samples [pos, pend)
            for (int ks = pos >> 2; ks <= (pend - 1) >> 2; ++ks) {
                const int ksamp = 4 * ks + lr;
                const bool in = ksamp >= pos && ksamp < pend;
                const double v = S.vy[lq * kMomLdk + ksamp];
                const double a = in ? v : 0.0;                 // A = VY: row p = l/4, k-slot = sample
                double b[NPT];                                 // B = VX^T: k-slot = sample, column q = 8 qt + l/4
#pragma unroll
                for (int qt = 0; qt < NPT; ++qt) b[qt] = S.vx[(8 * qt + lq) * kMomLdk + ksamp];
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const double ac = MAP ? a * S.beta[c * kMomLdk + ksamp] : a;   // the node weight rides on the delta powers
#pragma unroll
                    for (int qt = 0; qt < NPT; ++qt) dmma_m8n8k4(mt[c][qt][0], mt[c][qt][1], ac, b[qt]);
                }
            }
            pos = pend;
        }
        k += nb;
    }
    if (have) flush();
    queue_done(W, W.ctrl + (frames ? (long long)blockIdx.y * W.ctrl_stride : 0), item_id, lane);
}

}  // namespace e2e
