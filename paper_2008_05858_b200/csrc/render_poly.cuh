// render_poly.cuh -- steps a4 + a5 for the analytic PSF, sm_100a production kernel.
//
//   frame[j][i] += sum_k sum_t  BY_t[k][j] * AX_t[k][i]
//   AX_t[k][i] = w_k * FX_t,n(dx_k)   (n = i - X - nlo_x)      BY_t[k][j] = GY_t,n(dy_k)
//
// Work decomposition (one warp per work item, no block-level cooperation, no atomics):
//   item   = run of consecutive samples of one (fiber, order) strip (schedule built on the host, api.cu)
//   chunk  = maximal run of <= 32 consecutive samples inside one detector pixel: floor(x_k) = X, floor(y_k) = Y.
//            All its footprints (G9) lie in the fixed window  columns X + nlo_x .. , rows Y + nlo_y .. ,  and the
//            1-D pixel-integrated factors are polynomials of the sub-pixel phase (dx, dy) in [-1/2, 1/2)^2 whose
//            coefficients depend only on (t, n): poly_tables.h.  No special function is evaluated on the device.
//   The chunk's contraction over (k, t) is a dense fp64 GEMM (window rows x window columns x K = samples * terms).
//   It runs as mma.sync m8n8k4 f64 tiles: lane l evaluates exactly the fragment elements it owns,
//       B[k = l%4][n = l/4]  <- AX of column 8 ct + l/4 at sample 4 ks + l%4   (registers, never staged)
//       A[m = l/4][k = l%4]  <- BY of row    8 rt + l/4 at sample 4 ks + l%4   (staged once per term in shared memory)
//   so every polynomial is evaluated once and only the y-factors travel through shared memory.
//   The window is walked in panels of 24 x 24 pixels (3 x 3 tiles, 18 accumulator registers per lane); the
//   ESPRESSO-like and HIRES-like PSFs (footprint 23-24 px) need exactly one panel.
//   The finished panel is added to the frame by plain read-modify-write (ld.cg / st.cg): items that run in the
//   same launch never touch the same pixel, and a pixel's additions happen in a fixed order -> bit-reproducible.
#pragma once
#include "common.cuh"

namespace e2e {

constexpr int kPolyWarps = 4;          // warps per CTA
constexpr int kPanel = 24;             // panel edge in pixels (3 tiles of 8)
constexpr int kLdb = 28;               // leading dimension of the BY staging buffer (28 mod 16 = 12: conflict-free fragments)
constexpr int kMaxWin = 104;           // largest padded window edge (footprint limit 96 px + 2, padded to 8)


__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// per-warp shared-memory block
struct PolyWarpSmem {
    double by[32 * kLdb];              // BY[k][row of the panel]
    double dx[32], dy[32], w[32];      // sub-pixel phases and weights of the chunk's samples (0 beyond the chunk)
    unsigned colmask[kMaxWin];         // bit k: column n is inside sample k's footprint
    unsigned rowmask[kMaxWin];
};

template <int P>
__global__ void __launch_bounds__(kPolyWarps * 32)
render_poly_kernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ ws,
                   const Strip* __restrict__ strips, const Item* __restrict__ items, int n_items, PolyParam Q,
                   double* __restrict__ frame, int nx, int ny)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int item_id = blockIdx.x * kPolyWarps + warp;
    if (item_id >= n_items) return;
    PolyWarpSmem& S = reinterpret_cast<PolyWarpSmem*>(smem_raw)[warp];
    const Item it = items[item_id];
    const Strip st = strips[it.strip];
    const int lq = lane >> 2, lr = lane & 3;                  // fragment coordinates: l/4 and l%4
    for (int i = lane; i < 32 * kLdb; i += 32) S.by[i] = 0.0;  // tiles beyond the window read (and discard) these

    long long k = (long long)it.chunk0 * 32;
    long long kend = k + (long long)it.nchunks * 32;
    if (kend > st.n) kend = st.n;

    while (k < kend) {
        // ---- cut the next chunk: leading run of samples in the pixel of sample k
        const long long kk = k + lane;
        const bool valid = kk < kend;
        const long long kidx = st.off + (valid ? kk : kend - 1);
        const double xk = xs[kidx], yk = ys[kidx];
        const double wk = valid ? ws[kidx] : 0.0;
        const int fx = __double2int_rd(xk), fy = __double2int_rd(yk);
        const int X = __shfl_sync(0xffffffffu, fx, 0), Y = __shfl_sync(0xffffffffu, fy, 0);
        const unsigned same = __ballot_sync(0xffffffffu, valid && fx == X && fy == Y);
        const int nc = (same == 0xffffffffu) ? 32 : (__ffs(~same) - 1);      // lane 0 is always in
        k += nc;
        const bool in = lane < nc;
        // G9 footprint box of this lane's sample (same operations as the setup of the oracle's box)
        const int ilo = __double2int_ru(__dsub_rn(xk, Q.hbx)), ihi = __double2int_rd(__dadd_rn(xk, Q.hbx));
        const int jlo = __double2int_ru(__dsub_rn(yk, Q.hby)), jhi = __double2int_rd(__dadd_rn(yk, Q.hby));
        const bool act = in && wk != 0.0 && ihi >= 0 && ilo < nx && jhi >= 0 && jlo < ny && ihi >= ilo && jhi >= jlo;
        if (!__any_sync(0xffffffffu, act)) continue;
        // union of the active footprints, clipped to the detector: the only pixels this chunk may touch
        const int BIG = 0x3fffffff;
        int cmin = act ? ilo : BIG, cmax = act ? ihi : -BIG, rmin = act ? jlo : BIG, rmax = act ? jhi : -BIG;
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) {
            cmin = min(cmin, __shfl_xor_sync(0xffffffffu, cmin, s));
            cmax = max(cmax, __shfl_xor_sync(0xffffffffu, cmax, s));
            rmin = min(rmin, __shfl_xor_sync(0xffffffffu, rmin, s));
            rmax = max(rmax, __shfl_xor_sync(0xffffffffu, rmax, s));
        }
        cmin = max(cmin, 0); cmax = min(cmax, nx - 1); rmin = max(rmin, 0); rmax = min(rmax, ny - 1);
        const int c0 = X + Q.nlo_x, r0 = Y + Q.nlo_y;                        // window origin
        __syncwarp();                                                       // previous chunk's readers are done
        S.dx[lane] = in ? (xk - (double)X) - 0.5 : 0.0;
        S.dy[lane] = in ? (yk - (double)Y) - 0.5 : 0.0;
        S.w[lane] = act ? wk : 0.0;
        for (int c = 0; c < Q.ncol_pad; ++c) {
            const int col = c0 + c;
            const unsigned b = __ballot_sync(0xffffffffu, act && col >= ilo && col <= ihi);
            if (lane == (c & 31)) S.colmask[c] = b;
        }
        for (int r = 0; r < Q.nrow_pad; ++r) {
            const int row = r0 + r;
            const unsigned b = __ballot_sync(0xffffffffu, act && row >= jlo && row <= jhi);
            if (lane == (r & 31)) S.rowmask[r] = b;
        }
        __syncwarp();
        const int ksteps = (nc + 3) >> 2;

        for (int rp = 0; rp < Q.nrow_pad; rp += kPanel) {
            if (r0 + rp > rmax || r0 + rp + kPanel - 1 < rmin) continue;
            for (int cp = 0; cp < Q.ncol_pad; cp += kPanel) {
                if (c0 + cp > cmax || c0 + cp + kPanel - 1 < cmin) continue;
                double acc[9][2];
#pragma unroll
                for (int a = 0; a < 9; ++a) { acc[a][0] = 0.0; acc[a][1] = 0.0; }

                for (int t = 0; t < Q.T; ++t) {
                    // ---- y-factors of term t for the panel's rows -> shared memory (A fragments)
#pragma unroll 1
                    for (int rt = 0; rt < 3; ++rt) {
                        const int n = rp + 8 * rt + lq;
                        if (rp + 8 * rt >= Q.nrow_pad) break;                // warp-uniform
                        const double* cf = Q.ty + ((size_t)t * (P + 1)) * Q.nrow_pad + n;
                        double a[P + 1];
#pragma unroll
                        for (int p = 0; p <= P; ++p) a[p] = __ldg(cf + (size_t)p * Q.nrow_pad);
                        const unsigned rm = S.rowmask[n];
#pragma unroll 2
                        for (int ks = 0; ks < ksteps; ++ks) {
                            const int ksamp = 4 * ks + lr;
                            const double d = S.dy[ksamp];
                            double v = a[P];
#pragma unroll
                            for (int p = P - 1; p >= 0; --p) v = fma(v, d, a[p]);
                            S.by[ksamp * kLdb + 8 * rt + lq] = ((rm >> ksamp) & 1u) ? v : 0.0;
                        }
                    }
                    __syncwarp();
                    // ---- x-factors of term t in registers (B fragments) and the tile products
#pragma unroll 1
                    for (int ct = 0; ct < 3; ++ct) {
                        const int n = cp + 8 * ct + lq;
                        if (cp + 8 * ct >= Q.ncol_pad) break;                // warp-uniform
                        const double* cf = Q.tx + ((size_t)t * (P + 1)) * Q.ncol_pad + n;
                        double a[P + 1];
#pragma unroll
                        for (int p = 0; p <= P; ++p) a[p] = __ldg(cf + (size_t)p * Q.ncol_pad);
                        const unsigned cm = S.colmask[n];
#pragma unroll 2
                        for (int ks = 0; ks < ksteps; ++ks) {
                            const int ksamp = 4 * ks + lr;
                            const double d = S.dx[ksamp];
                            double v = a[P];
#pragma unroll
                            for (int p = P - 1; p >= 0; --p) v = fma(v, d, a[p]);
                            v *= S.w[ksamp];
                            const double b = ((cm >> ksamp) & 1u) ? v : 0.0;
                            const double* ap = &S.by[ksamp * kLdb + lq];
                            if (ct == 0) {
                                dmma_m8n8k4(acc[0][0], acc[0][1], ap[0], b);
                                dmma_m8n8k4(acc[3][0], acc[3][1], ap[8], b);
                                dmma_m8n8k4(acc[6][0], acc[6][1], ap[16], b);
                            } else if (ct == 1) {
                                dmma_m8n8k4(acc[1][0], acc[1][1], ap[0], b);
                                dmma_m8n8k4(acc[4][0], acc[4][1], ap[8], b);
                                dmma_m8n8k4(acc[7][0], acc[7][1], ap[16], b);
                            } else {
                                dmma_m8n8k4(acc[2][0], acc[2][1], ap[0], b);
                                dmma_m8n8k4(acc[5][0], acc[5][1], ap[8], b);
                                dmma_m8n8k4(acc[8][0], acc[8][1], ap[16], b);
                            }
                        }
                    }
                    __syncwarp();
                }
                // ---- a5: add the panel to the frame.  lane owns C[row 8 rt + l/4][cols 8 ct + 2 (l%4) + {0,1}]
#pragma unroll
                for (int rt = 0; rt < 3; ++rt) {
                    const int row = r0 + rp + 8 * rt + lq;
                    if (row < rmin || row > rmax) continue;
#pragma unroll
                    for (int ct = 0; ct < 3; ++ct) {
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int col = c0 + cp + 8 * ct + 2 * lr + e;
                            if (col < cmin || col > cmax) continue;
                            double* p = frame + (size_t)row * nx + col;
                            __stcg(p, __ldcg(p) + acc[rt * 3 + ct][e]);
                        }
                    }
                }
            }
        }
    }
}

}  // namespace e2e
