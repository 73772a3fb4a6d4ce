// render_tabcell.cuh -- steps a4 + a5 for the tabulated, field-dependent PSF: production kernel.
//
// T1-T3 of DESIGN.md ("ray tracing software to recover the complete PSF"; BJ config "Field-dependent PSF"):
// the kernel is a piecewise-constant density on 1/os-px cells, so its summed-area table C is piecewise bilinear and
// the pixel integral of one sample is a 4-corner difference of bilinear look-ups in C.  Two exact regroupings:
//
//  (1) difference first: PI[gy][gx] = sum of the kernel cells in [gy, gy+os) x [gx, gx+os) (clipped to the kernel)
//      is the pixel integral for a pixel whose lower-left corner sits ON the fine-grid point (gx, gy).  Differencing
//      commutes with the bilinear look-up, so for a pixel corner at fine-grid position (ex, ey) = (gx + 1 - fa, ...)
//          P = fa fb PI[gy][gx] + (1-fa) fb PI[gy][gx+1] + fa (1-fb) PI[gy+1][gx] + (1-fa)(1-fb) PI[gy+1][gx+1]
//      PI is built on the host in long double: no cancellation is left on the device.
//  (2) deposit first: all samples of a *cell* (same first column ilo, first row jlo, same 4 field nodes) address the
//      table at g = os n - a' for window column n and a sub-pixel offset index a' in 0..os that does not depend on n.
//      So their weights are summed once, cloud-in-cell on the 1/os-px grid and split over the 4 field nodes (T3, the
//      blend is linear):
//          W[c][b'][a'] = sum_k w_k beta_c(x_k, y_k) Fy_k[b'] Fx_k[a'],   Fx_k[A_k + 1] = fa_k, Fx_k[A_k] = 1 - fa_k
//      and the cell's frame contribution is   out[j][i] = sum_{c,b',a'} W[c][b'][a'] PI_c[os j - b'][os i - a'].
//      The table is stored phase-major, PI_c[ry][rx][J][I] with fine index + os = os J + ry, so that for one
//      (c, b', a') the window's pixels read a contiguous (npix+1) x (npix+1) block: coalesced, L1-resident.
//
// Per sample only the deposit is left (16 products); the table walk, (npix+1)^2 FMAs per non-zero weight, is paid
// once per cell (~32 samples at 32 samples/px).  One warp per work item (schedule of api.cu), no atomics, frame
// added by read-modify-write in a fixed order -> bit-reproducible.
#pragma once
#include "common.cuh"

namespace e2e {

#ifndef E2E_TC_WARPS
#define E2E_TC_WARPS 16
#endif
constexpr int kTcWarps = E2E_TC_WARPS;  // warps per CTA: one CTA per SM, its warps walk neighbouring runs of one strip (shared L1 working set)
constexpr int kTcMaxOs = 16;           // largest oversampling handled here (weight array (os+1)^2 x 4 per warp)
constexpr int kTcSlots = 8;            // pixels per lane and panel
constexpr int kTcPitch = 33;           // staging pitch: val[v][sample]

__host__ __device__ inline size_t tabcell_warp_smem_doubles(int os)
{
    return (size_t)4 * (os + 1) * (os + 1) + 16 * kTcPitch + 16;   // W | val | base (32 ints)
}

__global__ void __launch_bounds__(kTcWarps * 32)
render_tabcell_kernel(const double* __restrict__ xs, const double* __restrict__ ys, const double* __restrict__ ws,
                      const Strip* __restrict__ strips, const Item* __restrict__ items, int n_items, TabParam T,
                      double* __restrict__ frame, int nx, int ny)
{
    extern __shared__ double smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int item_id = blockIdx.x * kTcWarps + warp;
    if (item_id >= n_items) return;
    const int S = T.os + 1, S2 = S * S;
    double* Wt = smem + (size_t)warp * tabcell_warp_smem_doubles(T.os);   // [4][S][S]
    double* val = Wt + 4 * S2;                                            // [16][kTcPitch]
    int* base = reinterpret_cast<int*>(val + 16 * kTcPitch);              // [32]
    const Item it = items[item_id];
    const Strip st = strips[it.strip];
    const int ld = T.pi_ld, nwin = T.npix + 1, npx = nwin * nwin;
    const size_t node_stride = (size_t)T.os * T.os * ld * ld;
    const double dos = (double)T.os;

    for (int i = lane; i < 4 * S2; i += 32) Wt[i] = 0.0;
    // this lane's role in the deposit: v = lane & 15 -> (hy, hx, ey, ex)
    const int v = lane & 15;
    const int dep_off = (v >> 2) * S2 + ((v >> 1) & 1) * S + (v & 1);

    long long k = (long long)it.chunk0 * 32;
    long long kend = k + (long long)it.nchunks * 32;
    if (kend > st.n) kend = st.n;

    bool have = false, cell_nz = false;
    int cI = 0, cJ = 0, cG = 0, cH = 0;                       // cell key: first column / row, field node cell
    int aMin = 0, aMax = 0, bMin = 0, bMax = 0;               // range of sub-pixel offsets deposited in the open cell

    auto flush = [&]() {
        const bool dead = !cell_nz || cI + nwin <= 0 || cI >= nx || cJ + nwin <= 0 || cJ >= ny;
        if (!dead) {
            const int g1 = T.gx > 1 ? cG + 1 : cG, h1 = T.gy > 1 ? cH + 1 : cH;
            const double* node[4] = {T.pi + (size_t)(cH * T.gx + cG) * node_stride, T.pi + (size_t)(cH * T.gx + g1) * node_stride,
                                     T.pi + (size_t)(h1 * T.gx + cG) * node_stride, T.pi + (size_t)(h1 * T.gx + g1) * node_stride};
            for (int p0 = 0; p0 < npx; p0 += 32 * kTcSlots) {
                const int nslot = min(kTcSlots, (npx - p0 + 31) >> 5);
                double out[kTcSlots];
                int poff[kTcSlots];
#pragma unroll
                for (int s = 0; s < kTcSlots; ++s) {
                    const int p = p0 + lane + 32 * s;
                    const int j = p / nwin, i = p - j * nwin;
                    poff[s] = p < npx ? j * ld + i : 0;
                    out[s] = 0.0;
                }
                for (int c = 0; c < 4; ++c) {
                    const double* Pc = node[c];
                    if (c == 1 && T.gx == 1) continue;         // single-node axes: the second node carries no weight
                    if (c >= 2 && T.gy == 1) break;
                    for (int bp = bMin; bp <= bMax + 1; ++bp) {
                        const int ry = bp ? T.os - bp : 0, dJ = bp ? 0 : 1;
                        const double* Wrow = Wt + c * S2 + bp * S;
                        const double* Prow = Pc + ((size_t)(ry * T.os) * ld + dJ) * ld;
                        // no zero test inside: every offset of [aMin, aMax + 1] normally carries weight, and a
                        // branch-free body lets the table loads of consecutive offsets overlap
#pragma unroll 3
                        for (int ap = aMin; ap <= aMax + 1; ++ap) {
                            const double wv = Wrow[ap];
                            const int rx = ap ? T.os - ap : 0, dI = ap ? 0 : 1;
                            const double* src = Prow + (size_t)rx * ld * ld + dI;
#pragma unroll
                            for (int s = 0; s < kTcSlots; ++s)
                                if (s < nslot) out[s] = fma(wv, __ldg(src + poff[s]), out[s]);
                        }
                    }
                }
                // ---- a5
#pragma unroll
                for (int s = 0; s < kTcSlots; ++s) {
                    const int p = p0 + lane + 32 * s;
                    if (s < nslot && p < npx) {
                        const int j = p / nwin, i = p - j * nwin;
                        const int row = cJ + j, col = cI + i;
                        if (row >= 0 && row < ny && col >= 0 && col < nx) {
                            double* q = frame + (size_t)row * nx + col;
                            __stcg(q, __ldcg(q) + out[s]);
                        }
                    }
                }
            }
        }
        __syncwarp();
        for (int i = lane; i < 4 * S2; i += 32) Wt[i] = 0.0;
        __syncwarp();
    };

    while (k < kend) {
        const int nb = (int)min((long long)32, kend - k);
        const bool valid = lane < nb;
        const long long kidx = st.off + k + (valid ? lane : nb - 1);
        const double xk = xs[kidx], yk = ys[kidx];
        const double wk = valid ? ws[kidx] : 0.0;
        // G9 footprint box: first column / row (same operations as the oracle's box)
        const int ilo = __double2int_ru(__dsub_rn(xk, T.hb)), jlo = __double2int_ru(__dsub_rn(yk, T.hb));
        // sub-pixel phase in (0, 1] and its split on the 1/os grid
        const double tx = (((xk - (double)ilo) - T.c0) * dos), ty = (((yk - (double)jlo) - T.c0) * dos);
        const int A = min(max((int)ceil(tx) - 1, 0), T.os - 1), B = min(max((int)ceil(ty) - 1, 0), T.os - 1);
        const double fa = tx - (double)A, fb = ty - (double)B;
        // T3 field weights
        int g0 = 0, h0 = 0;
        double fx = 0.0, fy = 0.0;
        if (T.gx > 1) {
            const double t = fmin(fmax(xk * T.fsx, 0.0), (double)(T.gx - 1));
            g0 = min((int)floor(t), T.gx - 2);
            fx = t - (double)g0;
        }
        if (T.gy > 1) {
            const double t = fmin(fmax(yk * T.fsy, 0.0), (double)(T.gy - 1));
            h0 = min((int)floor(t), T.gy - 2);
            fy = t - (double)h0;
        }
        __syncwarp();                                          // previous batch's deposit readers are done
        {
            const double bx[2] = {1.0 - fx, fx}, by[2] = {1.0 - fy, fy};
            const double cx[2] = {1.0 - fa, fa}, cy[2] = {1.0 - fb, fb};
#pragma unroll
            for (int u = 0; u < 16; ++u)
                val[u * kTcPitch + lane] = wk * (by[u >> 3] * bx[(u >> 2) & 1]) * (cy[(u >> 1) & 1] * cx[u & 1]);
            base[lane] = B * S + A;
        }
        __syncwarp();
        int pos = 0;
        while (pos < nb) {
            const int kI = __shfl_sync(0xffffffffu, ilo, pos), kJ = __shfl_sync(0xffffffffu, jlo, pos);
            const int kG = __shfl_sync(0xffffffffu, g0, pos), kH = __shfl_sync(0xffffffffu, h0, pos);
            if (have && (kI != cI || kJ != cJ || kG != cG || kH != cH)) {
                flush();
                have = false;
            }
            if (!have) {
                have = true; cell_nz = false;
                cI = kI; cJ = kJ; cG = kG; cH = kH;
                aMin = bMin = 1 << 20; aMax = bMax = -1;
            }
            const unsigned same = __ballot_sync(0xffffffffu, valid && ilo == cI && jlo == cJ && g0 == cG && h0 == cH);
            const unsigned rest = ~(same >> pos);
            const int run = rest ? (__ffs(rest) - 1) : 32;
            const int pend = min(pos + run, nb);
            const bool in = lane >= pos && lane < pend;
            cell_nz = cell_nz || __any_sync(0xffffffffu, in && wk != 0.0);
            aMin = min(aMin, __reduce_min_sync(0xffffffffu, in ? A : (1 << 20)));
            aMax = max(aMax, __reduce_max_sync(0xffffffffu, in ? A : -1));
            bMin = min(bMin, __reduce_min_sync(0xffffffffu, in ? B : (1 << 20)));
            bMax = max(bMax, __reduce_max_sync(0xffffffffu, in ? B : -1));
            // ---- deposit, sample after sample (fixed order); lanes 0..15 own the 16 (node, corner) products
            if (lane < 16) {
                for (int s = pos; s < pend; ++s) {
                    const int idx = dep_off + base[s];
                    Wt[idx] += val[v * kTcPitch + s];
                }
            }
            __syncwarp();
            pos = pend;
        }
        k += nb;
    }
    if (have) flush();
}

}  // namespace e2e
