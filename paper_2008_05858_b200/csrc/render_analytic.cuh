// render_analytic.cuh -- steps a4 + a5 for the analytic PSF (uniform ellipse (x) gaussian), O4.
//
//   P(u, v) = sum_q wq * Ax_q(u) * By_q(v)           (Gauss-Chebyshev chord quadrature of the ellipse)
//   Ax_q(u) = Phi((u + 1/2 - s_q)/sx) - Phi((u - 1/2 - s_q)/sx)            pixel-integrated gaussian at chord abscissa s_q
//   By_q(v) = (sy / 2c_q) { [Psi(z+ + c/sy) - Psi(z+ - c/sy)] - [Psi(z- + c/sy) - Psi(z- - c/sy)] },  z+- = (v +- 1/2)/sy
//
// Work decomposition (one warp per work item, no block-level cooperation, no atomics):
//   item   = run of consecutive 32-sample chunks of one (fiber, order) strip
//   chunk  = 32 consecutive samples; lane <-> sample while the 1-D factors are evaluated ("edge phase"),
//            lane <-> 5x5 pixel patch of the chunk's pixel window while they are contracted ("outer-product phase").
//            The window is the union of the 32 footprints (<= 25 columns x 30 rows; larger unions are split).
//   The contraction over the chunk, frame[r][c] += sum_{k,q} By[q,k][r] * Ax[q,k][c], is a small dense fp64
//   GEMM (K = 32 samples x terms) fed from a warp-private shared-memory staging buffer; its result is added
//   to the frame by plain read-modify-write.  Items that run concurrently never touch the same pixel
//   (schedule built on the host: alternate runs of a strip in different launches, overlapping strips in
//   different launches), and every pixel's additions happen in a fixed order -> bit-reproducible.
#pragma once
#include "common.cuh"

namespace e2e {

constexpr int kWarpsPerCta = 4;
constexpr int kPatch = 5;          // 5 x 5 accumulators per lane
constexpr int kColGroups = 5;      // lanes 0..29: (row group 0..5) x (col group 0..4)
constexpr int kRowGroups = 6;
constexpr int kWinCols = kPatch * kColGroups;   // 25
constexpr int kWinRows = kPatch * kRowGroups;   // 30
constexpr int kLdk = 34;           // staging leading dimension (32 samples + 2: conflict-free 128-bit reads)

constexpr double kRsqrt2 = 0.70710678118654752440;
constexpr double kRsqrt2pi = 0.39894228040143267794;

// Phi(z) = flag + small, flag = [z >= 0], small = -+ erfc(|z|/sqrt2)/2: differences of Phi cancel the flags exactly
__device__ __forceinline__ void phi_split(double z, int& flag, double& small)
{
    double S = 0.5 * erfc(fabs(z) * kRsqrt2);
    flag = z >= 0.0;
    small = flag ? -S : S;
}
// Psi(-t) for t >= 0:  phi(t) - t * erfc(t/sqrt2)/2
__device__ __forceinline__ double psi_minus(double t)
{
    return fma(-t, 0.5 * erfc(t * kRsqrt2), exp(-0.5 * t * t) * kRsqrt2pi);
}
// E(z) = Psi(z + cs) - Psi(z - cs) = clamp(z + cs, 0, 2cs) + [Psi(-|z + cs|) - Psi(-|z - cs|)]
__device__ __forceinline__ double psi_span(double z, double cs)
{
    double lin = fmin(fmax(z + cs, 0.0), 2.0 * cs);
    return lin + (psi_minus(fabs(z + cs)) - psi_minus(fabs(z - cs)));
}

struct ChunkGeom {
    int ilo, ihi, jlo, jhi;
};

// smallest power-of-two split of the warp into segments whose union windows fit (wc x wr); returns segment length
__device__ __forceinline__ int segment_fit(bool act, const ChunkGeom& g, int wc, int wr, int& cmin, int& cmax, int& rmin,
                                           int& rmax)
{
    const int BIG = 0x3fffffff;
    int a = act ? g.ilo : BIG, b = act ? g.ihi : -BIG, c = act ? g.jlo : BIG, d = act ? g.jhi : -BIG;
    // full-warp butterfly first, then narrower ones while some segment does not fit
    for (int len = 32; len >= 1; len >>= 1) {
        int a2 = a, b2 = b, c2 = c, d2 = d;
        for (int s = len >> 1; s > 0; s >>= 1) {
            a2 = min(a2, __shfl_xor_sync(0xffffffffu, a2, s));
            b2 = max(b2, __shfl_xor_sync(0xffffffffu, b2, s));
            c2 = min(c2, __shfl_xor_sync(0xffffffffu, c2, s));
            d2 = max(d2, __shfl_xor_sync(0xffffffffu, d2, s));
        }
        bool ok = (b2 < a2) || ((b2 - a2 + 1 <= wc) && (d2 - c2 + 1 <= wr));
        if (__all_sync(0xffffffffu, ok) || len == 1) {
            cmin = a2; cmax = b2; rmin = c2; rmax = d2;
            return len;
        }
    }
    return 1;
}

__global__ void __launch_bounds__(kWarpsPerCta * 32)
render_analytic_kernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ ws,
                       const Strip* __restrict__ strips, const Item* __restrict__ items, int n_items,
                       AnalyticParam P, double* __restrict__ frame, int nx, int ny)
{
    extern __shared__ double smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int item_id = blockIdx.x * kWarpsPerCta + warp;
    if (item_id >= n_items) return;
    double* AX = smem + (size_t)warp * (kWinCols + kWinRows) * kLdk;   // [kWinCols][kLdk]
    double* BY = AX + kWinCols * kLdk;                                  // [kWinRows][kLdk]
    const Item it = items[item_id];
    const Strip st = strips[it.strip];
    const int rg = lane / kColGroups, cg = lane - rg * kColGroups;      // lanes 30, 31: rg = 6 (idle in the contraction)
    const bool worker = lane < kColGroups * kRowGroups;

    for (int c = it.chunk0; c < it.chunk0 + it.nchunks; ++c) {
        long long kk = (long long)c * 32 + lane;
        bool valid = kk < st.n;
        long long kidx = st.off + (valid ? kk : st.n - 1);
        double xk = xs[kidx], yk = ys[kidx], wk = valid ? ws[kidx] : 0.0;
        ChunkGeom g;
        g.ilo = __double2int_ru(__dsub_rn(xk, P.hbx));   // G9: ceil(x - hb) .. floor(x + hb)
        g.ihi = __double2int_rd(__dadd_rn(xk, P.hbx));
        g.jlo = __double2int_ru(__dsub_rn(yk, P.hby));
        g.jhi = __double2int_rd(__dadd_rn(yk, P.hby));
        bool act = valid && wk != 0.0 && g.ihi >= 0 && g.ilo < nx && g.jhi >= 0 && g.jlo < ny && g.ihi >= g.ilo && g.jhi >= g.jlo;
        if (!__any_sync(0xffffffffu, act)) continue;
        int cmin, cmax, rmin, rmax;
        // the staging buffer holds one 25 x 30 window; wider unions (large PSFs) are walked panel by panel
        int seglen = segment_fit(act, g, 4 * kWinCols, 4 * kWinRows, cmin, cmax, rmin, rmax);
        for (int seg0 = 0; seg0 < 32; seg0 += seglen) {
            // window of this segment (uniform inside the segment; take it from the segment's first lane)
            int c0 = __shfl_sync(0xffffffffu, cmin, seg0), c1 = __shfl_sync(0xffffffffu, cmax, seg0);
            int r0 = __shfl_sync(0xffffffffu, rmin, seg0), r1 = __shfl_sync(0xffffffffu, rmax, seg0);
            if (c1 < c0) continue;                                       // no active sample in this segment
            bool mine = act && lane >= seg0 && lane < seg0 + seglen;
            double wmine = mine ? wk : 0.0;
            for (int pr0 = r0; pr0 <= r1; pr0 += kWinRows) {
                for (int pc0 = c0; pc0 <= c1; pc0 += kWinCols) {
                    const int ncols = min(kWinCols, c1 - pc0 + 1), nrows = min(kWinRows, r1 - pr0 + 1);
                    double acc[kPatch][kPatch];
#pragma unroll
                    for (int u = 0; u < kPatch; ++u)
#pragma unroll
                        for (int t = 0; t < kPatch; ++t) acc[u][t] = 0.0;

                    for (int term = 0; term < P.n_terms; ++term) {
                        // ---- edge phase, x: Ax[col][lane] = w_k * wq * (F(e+1) - F(e)), F = Phi(. - s) (+ Phi(. + s))
                        {
                            const double s = P.s[term];
                            const bool paired = (P.paired >> term) & 1u;
                            const double scale = wmine * P.wq[term];
                            double d = (double)pc0 - 0.5 - xk;
                            int f0, f1; double s0, s1;
                            phi_split((d - s) * P.inv_sx, f0, s0);
                            if (paired) { int fb; double sb; phi_split((d + s) * P.inv_sx, fb, sb); f0 += fb; s0 += sb; }
                            for (int e = 0; e < ncols; ++e) {
                                d += 1.0;
                                phi_split((d - s) * P.inv_sx, f1, s1);
                                if (paired) { int fb; double sb; phi_split((d + s) * P.inv_sx, fb, sb); f1 += fb; s1 += sb; }
                                int col = pc0 + e;
                                double v = (col >= g.ilo && col <= g.ihi) ? scale * ((double)(f1 - f0) + (s1 - s0)) : 0.0;
                                AX[e * kLdk + lane] = v;
                                f0 = f1; s0 = s1;
                            }
                        }
                        // ---- edge phase, y: By[row][lane]
                        {
                            const double gsc = P.g[term];
                            double z = ((double)pr0 - 0.5 - yk) * P.inv_sy;
                            if (P.by_gauss) {
                                int f0, f1; double s0, s1;
                                phi_split(z, f0, s0);
                                for (int r = 0; r < nrows; ++r) {
                                    z = ((double)(pr0 + r) + 0.5 - yk) * P.inv_sy;
                                    phi_split(z, f1, s1);
                                    int row = pr0 + r;
                                    BY[r * kLdk + lane] = (row >= g.jlo && row <= g.jhi) ? ((double)(f1 - f0) + (s1 - s0)) : 0.0;
                                    f0 = f1; s0 = s1;
                                }
                            } else {
                                const double cs = P.cs[term];
                                double e0 = psi_span(z, cs), e1;
                                for (int r = 0; r < nrows; ++r) {
                                    z = ((double)(pr0 + r) + 0.5 - yk) * P.inv_sy;
                                    e1 = psi_span(z, cs);
                                    int row = pr0 + r;
                                    BY[r * kLdk + lane] = (row >= g.jlo && row <= g.jhi) ? gsc * (e1 - e0) : 0.0;
                                    e0 = e1;
                                }
                            }
                        }
                        __syncwarp();
                        // ---- outer-product phase: acc[u][t] += By[rg + 6u][k] * Ax[cg + 5t][k] over the segment's samples
                        if (worker) {
                            const int kb = seg0 & ~1, ke = seg0 + seglen;
                            for (int k2 = kb; k2 < ke; k2 += 2) {
                                double2 a[kPatch], b[kPatch];
#pragma unroll
                                for (int t = 0; t < kPatch; ++t)
                                    a[t] = *reinterpret_cast<const double2*>(&AX[(cg + kColGroups * t) * kLdk + k2]);
#pragma unroll
                                for (int u = 0; u < kPatch; ++u)
                                    b[u] = *reinterpret_cast<const double2*>(&BY[(rg + kRowGroups * u) * kLdk + k2]);
#pragma unroll
                                for (int u = 0; u < kPatch; ++u)
#pragma unroll
                                    for (int t = 0; t < kPatch; ++t) {
                                        acc[u][t] = fma(b[u].x, a[t].x, acc[u][t]);
                                        acc[u][t] = fma(b[u].y, a[t].y, acc[u][t]);
                                    }
                            }
                        }
                        __syncwarp();
                    }
                    // ---- a5: add the window into the frame (G11: pixels outside the detector are dropped)
                    if (worker) {
#pragma unroll
                        for (int u = 0; u < kPatch; ++u) {
                            int rr = rg + kRowGroups * u, row = pr0 + rr;
                            if (rr >= nrows || row < 0 || row >= ny) continue;
#pragma unroll
                            for (int t = 0; t < kPatch; ++t) {
                                int cc = cg + kColGroups * t, col = pc0 + cc;
                                if (cc >= ncols || col < 0 || col >= nx) continue;
                                size_t p = (size_t)row * nx + col;
                                frame[p] += acc[u][t];
                            }
                        }
                    }
                }
            }
        }
    }
}

}  // namespace e2e
