// render_tabulated.cuh -- steps a4 + a5 for the tabulated, field-dependent PSF (O5 / T1-T3).
//
// P:61 "ray tracing software to recover the complete PSF"; BASELINE.json config "Field-dependent PSF".
// T1  each kernel is (npix*os)^2 cell values = a piecewise-constant density on 1/os-px cells around the sample
// T2  pixel integral = sum of cell value x overlap.  The summed-area table C of the cells is piecewise
//     bilinear, so the integral over [x0,x1]x[y0,y1] is the 4-corner difference of bilinear lookups in C.
//     All pixel edges of one sample sit on a unit lattice, so the lookups are done once per lattice point.
// T3  field dependence: bilinear blend of the 4 surrounding node kernels at (x_k, y_k) (linear -> blend the lookups).
//
// Same warp-per-item decomposition as the analytic kernel; here lane <-> pixels of the chunk window and the
// samples of the chunk are walked one after the other (the PSF is not separable, so there is no GEMM form).
#pragma once
#include "common.cuh"
#include "render_analytic.cuh"

namespace e2e {

constexpr int kTabWin = 16;                 // window panel 16 x 16 pixels, 8 accumulators per lane
constexpr int kTabAcc = kTabWin * kTabWin / 32;

__device__ __forceinline__ double sat_bilinear(const double* __restrict__ S, int ld, int ia, int ib, double fa, double fb)
{
    const double* p = S + (size_t)ib * ld + ia;
    double v00 = __ldg(p), v01 = __ldg(p + 1), v10 = __ldg(p + ld), v11 = __ldg(p + ld + 1);
    double top = fma(fa, v01 - v00, v00), bot = fma(fa, v11 - v10, v10);
    return fma(fb, bot - top, top);
}

__global__ void __launch_bounds__(kWarpsPerCta * 32)
render_tabulated_kernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ ws,
                        const Strip* __restrict__ strips, const Item* __restrict__ items, int n_items,
                        TabParam T, int lat_ld, double* __restrict__ frame, int nx, int ny)
{
    extern __shared__ double smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int item_id = blockIdx.x * kWarpsPerCta + warp;
    if (item_id >= n_items) return;
    double* LAT = smem + (size_t)warp * lat_ld * lat_ld;      // [npix + 2][lat_ld] lattice of blended SAT lookups
    const Item it = items[item_id];
    const Strip st = strips[it.strip];
    const size_t tab_stride = (size_t)T.ld * T.ld;

    for (int c = it.chunk0; c < it.chunk0 + it.nchunks; ++c) {
        long long kk = (long long)c * 32 + lane;
        bool valid = kk < st.n;
        long long kidx = st.off + (valid ? kk : st.n - 1);
        double xk = xs[kidx], yk = ys[kidx], wk = valid ? ws[kidx] : 0.0;
        ChunkGeom g;
        g.ilo = __double2int_ru(__dsub_rn(xk, T.hb));
        g.ihi = __double2int_rd(__dadd_rn(xk, T.hb));
        g.jlo = __double2int_ru(__dsub_rn(yk, T.hb));
        g.jhi = __double2int_rd(__dadd_rn(yk, T.hb));
        bool act = valid && wk != 0.0 && g.ihi >= 0 && g.ilo < nx && g.jhi >= 0 && g.jlo < ny;
        unsigned actmask = __ballot_sync(0xffffffffu, act);
        if (!actmask) continue;
        // T3: field weights of this lane's sample
        int g0 = 0, h0 = 0; double fx = 0.0, fy = 0.0;
        if (T.gx > 1) {
            double tx = fmin(fmax(xk * T.fsx, 0.0), (double)(T.gx - 1));
            g0 = min((int)floor(tx), T.gx - 2);
            fx = tx - (double)g0;
        }
        if (T.gy > 1) {
            double ty = fmin(fmax(yk * T.fsy, 0.0), (double)(T.gy - 1));
            h0 = min((int)floor(ty), T.gy - 2);
            fy = ty - (double)h0;
        }
        int cmin, cmax, rmin, rmax;
        segment_fit(act, g, 1 << 20, 1 << 20, cmin, cmax, rmin, rmax);   // whole-chunk union; panels walk it
        for (int pr0 = rmin; pr0 <= rmax; pr0 += kTabWin) {
            for (int pc0 = cmin; pc0 <= cmax; pc0 += kTabWin) {
                double acc[kTabAcc];
#pragma unroll
                for (int a = 0; a < kTabAcc; ++a) acc[a] = 0.0;
                for (unsigned m = actmask; m; m &= m - 1) {
                    const int src = __ffs(m) - 1;
                    const double sx = __shfl_sync(0xffffffffu, xk, src), sy = __shfl_sync(0xffffffffu, yk, src);
                    const double sw = __shfl_sync(0xffffffffu, wk, src);
                    const int ilo = __shfl_sync(0xffffffffu, g.ilo, src), ihi = __shfl_sync(0xffffffffu, g.ihi, src);
                    const int jlo = __shfl_sync(0xffffffffu, g.jlo, src), jhi = __shfl_sync(0xffffffffu, g.jhi, src);
                    const int sg0 = __shfl_sync(0xffffffffu, g0, src), sh0 = __shfl_sync(0xffffffffu, h0, src);
                    const double sfx = __shfl_sync(0xffffffffu, fx, src), sfy = __shfl_sync(0xffffffffu, fy, src);
                    // footprint of this sample inside the panel
                    const int a0 = max(ilo, pc0), a1 = min(ihi, pc0 + kTabWin - 1);
                    const int b0 = max(jlo, pr0), b1 = min(jhi, pr0 + kTabWin - 1);
                    if (a1 < a0 || b1 < b0) continue;
                    const int na = a1 - a0 + 2, nb = b1 - b0 + 2;           // lattice points (pixel edges)
                    const int g1 = T.gx > 1 ? sg0 + 1 : sg0, h1 = T.gy > 1 ? sh0 + 1 : sh0;
                    const double* S00 = T.sat + (size_t)(sh0 * T.gx + sg0) * tab_stride;
                    const double* S01 = T.sat + (size_t)(sh0 * T.gx + g1) * tab_stride;
                    const double* S10 = T.sat + (size_t)(h1 * T.gx + sg0) * tab_stride;
                    const double* S11 = T.sat + (size_t)(h1 * T.gx + g1) * tab_stride;
                    const double w00 = (1.0 - sfy) * (1.0 - sfx), w01 = (1.0 - sfy) * sfx;
                    const double w10 = sfy * (1.0 - sfx), w11 = sfy * sfx;
                    for (int p = lane; p < na * nb; p += 32) {
                        const int b = p / na, a = p - b * na;
                        // edge position in cell units, clamped to the kernel extent (the SAT is constant outside)
                        double su = fmin(fmax((((double)(a0 + a) - 0.5 - sx) + T.half) * (double)T.os, 0.0), (double)T.n);
                        double sv = fmin(fmax((((double)(b0 + b) - 0.5 - sy) + T.half) * (double)T.os, 0.0), (double)T.n);
                        int ia = min((int)su, T.n - 1), ib = min((int)sv, T.n - 1);
                        double fa = su - (double)ia, fb = sv - (double)ib;
                        double v = w00 * sat_bilinear(S00, T.ld, ia, ib, fa, fb);
                        if (w01 != 0.0) v = fma(w01, sat_bilinear(S01, T.ld, ia, ib, fa, fb), v);
                        if (w10 != 0.0) v = fma(w10, sat_bilinear(S10, T.ld, ia, ib, fa, fb), v);
                        if (w11 != 0.0) v = fma(w11, sat_bilinear(S11, T.ld, ia, ib, fa, fb), v);
                        LAT[b * lat_ld + a] = v;
                    }
                    __syncwarp();
#pragma unroll
                    for (int q = 0; q < kTabAcc; ++q) {
                        const int pix = lane + 32 * q;                      // pixel of the panel: row pix / 16, col pix % 16
                        const int col = pc0 + (pix & (kTabWin - 1)), row = pr0 + (pix >> 4);
                        if (col >= a0 && col <= a1 && row >= b0 && row <= b1) {
                            const int a = col - a0, b = row - b0;
                            double v = (LAT[(b + 1) * lat_ld + a + 1] - LAT[b * lat_ld + a + 1]) -
                                       (LAT[(b + 1) * lat_ld + a] - LAT[b * lat_ld + a]);
                            acc[q] = fma(sw, v, acc[q]);
                        }
                    }
                    __syncwarp();
                }
#pragma unroll
                for (int q = 0; q < kTabAcc; ++q) {
                    const int pix = lane + 32 * q;
                    const int col = pc0 + (pix & (kTabWin - 1)), row = pr0 + (pix >> 4);
                    if (col <= cmax && row <= rmax && col >= 0 && col < nx && row >= 0 && row < ny) {
                        double* p = frame + (size_t)row * nx + col;
                        __stcg(p, __ldcg(p) + acc[q]);
                    }
                }
            }
        }
    }
}

}  // namespace e2e
