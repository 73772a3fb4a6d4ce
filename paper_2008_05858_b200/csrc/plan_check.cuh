// plan_check.cuh -- device-side verification of the render schedule (e2e_plan_check; test hook, not on the render path).
//
// The frame is accumulated with L2 reductions, so its bits are reproducible only if every pixel's additions happen in a
// fixed order.  That rests on invariants of the HOST schedule (api.cu build_plan); the kernels below check
// them on the real geometry, pixel by pixel, by stamping the footprint boxes (G9) of every item into an owner frame:
//
//   (1) phase launches (render_poly / render_analytic / render_tabcell / render_tabulated): no two items of one phase
//       share a pixel;
//   (2) queue launch (render_moment): run under the SAME queue discipline as the render kernel (queue_take / queue_done:
//       atomic ticket, wait for the dependency counter, release the successors), every item swaps its id into the owner frame; the previous owner of a pixel
//       must be one of the item's direct dependencies (or the item itself, or nobody).  If any two items that share a
//       pixel were not ordered by an edge, the write sequence of that pixel would contain a consecutive pair without an
//       edge in ANY execution, so one run with zero violations proves that every pixel's writers form a chain;
//   (3) row bands (host path; the 2-band device path of the phase-launched kernels): bands share no pixel, and a band
//       writes no row that an earlier band's copy to the host has already declared final.
#pragma once
#include "common.cuh"
#include "setup.cuh"
#include "render_moment.cuh"

namespace e2e {

struct PlanCheckCounters {
    unsigned long long claimed;        // first claims of a pixel
    unsigned long long conflicts;      // claims that found a foreign owner the rule does not allow
    unsigned long long early_rows;     // pixels above the band's first allowed row
};

// footprint box of sample k of strip (fiber, order), clipped to the detector; same operations as the render kernels
__device__ __forceinline__ void sample_box(const FormatView& f, int fiber, int o, long long k, double hbx, double hby, int nx, int ny,
                                           int& i0, int& i1, int& j0, int& j1)
{
    double lam, X, Y;
    sample_position_fast(f, o, k, lam, X, Y);
    const double xk = __dadd_rn(X, f.fiber_dx[fiber]), yk = __dadd_rn(Y, f.fiber_dy[fiber]);
    i0 = max(__double2int_ru(__dsub_rn(xk, hbx)), 0); i1 = min(__double2int_rd(__dadd_rn(xk, hbx)), nx - 1);
    j0 = max(__double2int_ru(__dsub_rn(yk, hby)), 0); j1 = min(__double2int_rd(__dadd_rn(yk, hby)), ny - 1);
}

// mode 0: phase launch -- one warp per item of items[0 .. n), id = item index + 1, a foreign owner is a conflict
// mode 1: band stamp   -- id = band + 1 for every item, a foreign owner is a conflict; rows < min_row are counted
// mode 2: persistent   -- queue discipline of render_moment_kernel; the previous owner must be a direct dependency
__global__ void __launch_bounds__(32) plan_check_kernel(FormatView f, const Strip* __restrict__ strips, const Item* __restrict__ items,
                                                        int n, int mode, int band_id, int min_row, QueueParam W, double hbx, double hby,
                                                        int* __restrict__ owner, PlanCheckCounters* __restrict__ cnt)
{
    const int lane = threadIdx.x & 31;
    const int nx = f.nx, ny = f.ny;
    for (int q = blockIdx.x;; q += gridDim.x) {
        int item_id;
        if (mode == 2) {
            item_id = queue_take(W, W.ctrl, lane);
            if (item_id < 0) break;
        } else {
            if (q >= n) break;
            item_id = q;
        }
        const Item it = items[item_id];
        const Strip st = strips[it.strip];
        const int fiber = it.strip / f.n_orders, o = it.strip - fiber * f.n_orders;
        const int my = mode == 1 ? band_id + 1 : item_id + 1;
        long long k = (long long)it.chunk0 * 32;
        long long kend = k + (long long)it.nchunks * 32;
        if (kend > st.n) kend = st.n;
        int pI0 = 1, pI1 = 0, pJ0 = 1, pJ1 = 0;                  // box of the sample before this batch (none yet)
        unsigned long long claimed = 0, conflicts = 0, early = 0;
        while (k < kend) {
            const int nb = (int)min((long long)32, kend - k);
            int i0, i1, j0, j1;
            sample_box(f, fiber, o, k + min(lane, nb - 1), hbx, hby, nx, ny, i0, i1, j0, j1);
            // stamp a box only where it differs from the previous sample's (consecutive samples share their box)
            int qi0 = __shfl_up_sync(0xffffffffu, i0, 1), qi1 = __shfl_up_sync(0xffffffffu, i1, 1);
            int qj0 = __shfl_up_sync(0xffffffffu, j0, 1), qj1 = __shfl_up_sync(0xffffffffu, j1, 1);
            if (lane == 0) { qi0 = pI0; qi1 = pI1; qj0 = pJ0; qj1 = pJ1; }
            unsigned fresh = __ballot_sync(0xffffffffu, lane < nb && (i0 != qi0 || i1 != qi1 || j0 != qj0 || j1 != qj1));
            while (fresh) {
                const int src = __ffs(fresh) - 1;
                fresh &= fresh - 1;
                const int bi0 = __shfl_sync(0xffffffffu, i0, src), bi1 = __shfl_sync(0xffffffffu, i1, src);
                const int bj0 = __shfl_sync(0xffffffffu, j0, src), bj1 = __shfl_sync(0xffffffffu, j1, src);
                const int bw = bi1 - bi0 + 1, bh = bj1 - bj0 + 1;
                if (bw <= 0 || bh <= 0) continue;
                for (int t = lane; t < bw * bh; t += 32) {
                    const int row = bj0 + t / bw, col = bi0 + t % bw;
                    int* cell = owner + (size_t)row * nx + col;
                    if (mode == 2) {
                        const int prev = atomicExch(cell, my);
                        if (prev == 0) ++claimed;
                        else if (prev != my) {
                            bool ok = false;
                            for (int d = W.dep_off[item_id]; d < W.dep_off[item_id + 1] && !ok; ++d) ok = W.dep_idx[d] + 1 == prev;
                            if (!ok) ++conflicts;
                        }
                    } else {
                        const int prev = atomicCAS(cell, 0, my);
                        if (prev == 0) ++claimed;
                        else if (prev != my) ++conflicts;
                        if (mode == 1 && row < min_row) ++early;
                    }
                }
            }
            pI0 = __shfl_sync(0xffffffffu, i0, nb - 1); pI1 = __shfl_sync(0xffffffffu, i1, nb - 1);
            pJ0 = __shfl_sync(0xffffffffu, j0, nb - 1); pJ1 = __shfl_sync(0xffffffffu, j1, nb - 1);
            k += nb;
        }
        for (int s = 16; s > 0; s >>= 1) {
            claimed += __shfl_xor_sync(0xffffffffu, claimed, s);
            conflicts += __shfl_xor_sync(0xffffffffu, conflicts, s);
            early += __shfl_xor_sync(0xffffffffu, early, s);
        }
        if (lane == 0) {
            if (claimed) atomicAdd(&cnt->claimed, claimed);
            if (conflicts) atomicAdd(&cnt->conflicts, conflicts);
            if (early) atomicAdd(&cnt->early_rows, early);
        }
        if (mode == 2) queue_done(W, W.ctrl, item_id, lane);
    }
}

}  // namespace e2e
