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
// once per cell (~32 samples at 32 samples/px).
//  (3) groups: up to kTcGroup consecutive cells of a strip that differ only in ilo read the SAME table entries (their
//      windows are shifted by whole pixels), so the walk loads each entry once and feeds one accumulator set per cell;
//      the shifted windows are summed in a warp-private shared tile and reach the frame with one L2 reduction per pixel.
// One warp per work item (schedule of api.cu), fixed order everywhere (the reductions of successive groups are ordered
// by the flush's __syncwarp()) -> bit-reproducible.
#pragma once
#include "common.cuh"

namespace e2e {

#ifndef E2E_TC_WARPS
#define E2E_TC_WARPS 16
#endif
constexpr int kTcWarps = E2E_TC_WARPS;  // warps per CTA: one CTA per SM, its warps walk neighbouring runs of one strip (shared L1 working set)
constexpr int kTcMaxOs = 16;           // largest oversampling handled here (weight array per warp)
constexpr int kTcSlots = 5;            // pixels per lane and panel (160 px: the 12 x 12 window of an 11-px kernel in one panel)
#ifndef E2E_TC_GROUP
#define E2E_TC_GROUP 4
#endif
constexpr int kTcGroup = E2E_TC_GROUP;            // cells per group (power of two)
constexpr int kTcRows = 4;             // weight rows per group: b' - (B0 - 1) in 0..3
constexpr int kTcPitch = 33;           // staging pitch: [value][sample]
// shared tile of a single-panel group: 12 rows x (12 + kTcGroup - 1) columns for the largest window that fits one panel.  Not a
// double more than needed: at 16 warps the CTA then takes 130 KB of shared memory, under the 132-KB carve-out step, which leaves
// the L1 124 KB instead of 92 KB for the table slices (6.94 -> 6.82 ms per field_psf frame)
constexpr int kTcTile = 12 * (12 + kTcGroup - 1) + 4;

__host__ __device__ inline size_t tabcell_warp_smem_doubles(int os)
{
    // W[group slot][node][row][os + 1] | wb[4][pitch] | cc[4][pitch] | base (32 ints) | tile
    return (size_t)kTcGroup * 4 * kTcRows * (os + 1) + 8 * kTcPitch + 16 + kTcTile;
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
    const int S = T.os + 1, SR = kTcRows * S, SN = 4 * SR, nW = kTcGroup * SN;
    double* Wt = smem + (size_t)warp * tabcell_warp_smem_doubles(T.os);   // [slot][node][row][S]
    double* wb = Wt + nW;                                                 // [4][pitch]  w * beta_node
    double* cc = wb + 4 * kTcPitch;                                       // [4][pitch]  Fy[ey] * Fx[ex]
    int* base = reinterpret_cast<int*>(cc + 4 * kTcPitch);                // [32]        B * S + A
    double* tile = cc + 4 * kTcPitch + 16;                                // [nwin][nwin + kTcGroup - 1]
    const Item it = items[item_id];
    const Strip st = strips[it.strip];
    const int ld = T.pi_ld, nwin = T.npix + 1, npx = nwin * nwin;
    const size_t node_stride = (size_t)T.os * T.os * ld * ld;
    const double dos = (double)T.os;
    const int tpitch = nwin + kTcGroup - 1;
    // groups need the whole window in one panel and the summed tile in shared memory; larger kernels run cell by cell
    const int max_cells = (npx <= 32 * kTcSlots && nwin * tpitch <= kTcTile) ? kTcGroup : 1;

    for (int i = lane; i < nW; i += 32) Wt[i] = 0.0;
    // this lane's role in the deposit: v = lane & 15 -> (hy, hx, ey, ex)
    const int v = lane & 15;
    const int dep_off = (v >> 2) * SR + ((v >> 1) & 1) * S + (v & 1);

    long long k = (long long)it.chunk0 * 32;
    long long kend = k + (long long)it.nchunks * 32;
    if (kend > st.n) kend = st.n;

    bool have = false, grp_nz = false;
    int gI0 = 0, gJ = 0, gG = 0, gH = 0, gB0 = 0;             // group key: first cell's column, row, field node cell, y-offset bin
    int mMin = 0, mMax = 0;                                    // member cells: ilo - gI0 in [mMin, mMax]
    int aMin = 0, aMax = 0, rMin = 0, rMax = 0;                // x offsets / weight rows deposited in the open group

    auto flush = [&]() {
        const int ncell = mMax - mMin + 1, c0col = gI0 + mMin;
        const bool dead = !grp_nz || c0col + nwin + ncell - 1 <= 0 || c0col >= nx || gJ + nwin <= 0 || gJ >= ny;
        if (!dead) {
            const int g1 = T.gx > 1 ? gG + 1 : gG, h1 = T.gy > 1 ? gH + 1 : gH;
            const double* node[4] = {T.pi + (size_t)(gH * T.gx + gG) * node_stride, T.pi + (size_t)(gH * T.gx + g1) * node_stride,
                                     T.pi + (size_t)(h1 * T.gx + gG) * node_stride, T.pi + (size_t)(h1 * T.gx + g1) * node_stride};
            int wslot[kTcGroup];                               // weight slot of member g (rotating: (ilo - gI0) & 3)
#pragma unroll
            for (int g = 0; g < kTcGroup; ++g) wslot[g] = ((mMin + g) & (kTcGroup - 1)) * SN;
            for (int p0 = 0; p0 < npx; p0 += 32 * kTcSlots) {
                const int nslot = min(kTcSlots, (npx - p0 + 31) >> 5);
                double out[kTcGroup][kTcSlots];
                int poff[kTcSlots];
#pragma unroll
                for (int s = 0; s < kTcSlots; ++s) {
                    const int p = p0 + lane + 32 * s;
                    const int j = p / nwin, i = p - j * nwin;
                    poff[s] = p < npx ? j * ld + i : 0;
#pragma unroll
                    for (int g = 0; g < kTcGroup; ++g) out[g][s] = 0.0;
                }
                for (int c = 0; c < 4; ++c) {
                    if (c == 1 && T.gx == 1) continue;         // single-node axes: the second node carries no weight
                    if (c >= 2 && T.gy == 1) break;
                    const double* Pc = node[c];
                    for (int rb = rMin; rb <= rMax + 1; ++rb) {
                        const int bp = gB0 - 1 + rb;           // b' in 0..os
                        const int ry = bp ? T.os - bp : 0, dJ = bp ? 0 : 1;
                        const double* Wrow = Wt + c * SR + rb * S;
                        const double* Prow = Pc + ((size_t)(ry * T.os) * ld + dJ) * ld;
                        // branch-free body: the table loads of consecutive offsets overlap
#pragma unroll 9
                        for (int ap = aMin; ap <= aMax + 1; ++ap) {
                            double wv[kTcGroup];
#pragma unroll
                            for (int g = 0; g < kTcGroup; ++g) wv[g] = Wrow[wslot[g] + ap];
                            const int rx = ap ? T.os - ap : 0, dI = ap ? 0 : 1;
                            const double* src = Prow + (size_t)rx * ld * ld + dI;
#pragma unroll
                            for (int s = 0; s < kTcSlots; ++s)
                                if (s < nslot) {
                                    const double pv = __ldg(src + poff[s]);
#pragma unroll
                                    for (int g = 0; g < kTcGroup; ++g) out[g][s] = fma(wv[g], pv, out[g][s]);
                                }
                        }
                    }
                }
                // ---- a5
                if (max_cells > 1) {
                    // single panel: sum the members' shifted windows in the shared tile, then one pass over the frame
                    const int ncol = nwin + ncell - 1, ntile = nwin * ncol;
                    for (int q = lane; q < ntile; q += 32) tile[q] = 0.0;
                    __syncwarp();
#pragma unroll
                    for (int g = 0; g < kTcGroup; ++g) {
                        if (g < ncell) {
#pragma unroll
                            for (int s = 0; s < kTcSlots; ++s) {
                                const int p = lane + 32 * s;
                                if (s < nslot && p < npx) {
                                    const int j = p / nwin, i = p - j * nwin;
                                    tile[j * ncol + g + i] += out[g][s];
                                }
                            }
                            __syncwarp();
                        }
                    }
                    for (int q = lane; q < ntile; q += 32) {
                        const int j = q / ncol, i = q - j * ncol;
                        const int row = gJ + j, col = c0col + i;
                        if (row >= 0 && row < ny && col >= 0 && col < nx) {
                            double* dst = frame + (size_t)row * nx + col;
                            atomicAdd(dst, tile[q]);        // L2 reduction, no round trip; ordered by the flush's __syncwarp()
                        }
                    }
                } else {
#pragma unroll
                    for (int s = 0; s < kTcSlots; ++s) {
                        const int p = p0 + lane + 32 * s;
                        if (s < nslot && p < npx) {
                            const int j = p / nwin, i = p - j * nwin;
                            const int row = gJ + j, col = c0col + i;
                            if (row >= 0 && row < ny && col >= 0 && col < nx) {
                                double* dst = frame + (size_t)row * nx + col;
                                atomicAdd(dst, out[0][s]);
                            }
                        }
                    }
                }
            }
        }
        __syncwarp();
        for (int i = lane; i < nW; i += 32) Wt[i] = 0.0;
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
            for (int u = 0; u < 4; ++u) {
                wb[u * kTcPitch + lane] = wk * (by[u >> 1] * bx[u & 1]);
                cc[u * kTcPitch + lane] = cy[u >> 1] * cx[u & 1];
            }
            base[lane] = B * S + A;
        }
        __syncwarp();
        int pos = 0;
        while (pos < nb) {
            const int kI = __shfl_sync(0xffffffffu, ilo, pos), kJ = __shfl_sync(0xffffffffu, jlo, pos);
            const int kG = __shfl_sync(0xffffffffu, g0, pos), kH = __shfl_sync(0xffffffffu, h0, pos);
            const int kB = __shfl_sync(0xffffffffu, B, pos);
            if (have) {
                const int m = kI - gI0;
                const bool fits = kJ == gJ && kG == gG && kH == gH && kB >= gB0 - 1 && kB <= gB0 + 1 &&
                                  max(mMax, m) - min(mMin, m) < max_cells;
                if (!fits) {
                    flush();
                    have = false;
                }
            }
            if (!have) {
                have = true; grp_nz = false;
                gI0 = kI; gJ = kJ; gG = kG; gH = kH; gB0 = kB;
                mMin = mMax = 0;
                aMin = rMin = 1 << 20; aMax = rMax = -1;
            }
            const int m = kI - gI0;
            mMin = min(mMin, m); mMax = max(mMax, m);
            const int rbs = B - gB0 + 1;                       // weight row of this lane's sample (ey = 0)
            const unsigned same = __ballot_sync(0xffffffffu, valid && ilo == kI && jlo == gJ && g0 == gG && h0 == gH &&
                                                                 rbs >= 0 && rbs <= 2);
            const unsigned rest = ~(same >> pos);
            const int run = rest ? (__ffs(rest) - 1) : 32;
            const int pend = min(pos + run, nb);
            const bool in = lane >= pos && lane < pend;
            grp_nz = grp_nz || __any_sync(0xffffffffu, in && wk != 0.0);
            aMin = min(aMin, __reduce_min_sync(0xffffffffu, in ? A : (1 << 20)));
            aMax = max(aMax, __reduce_max_sync(0xffffffffu, in ? A : -1));
            rMin = min(rMin, __reduce_min_sync(0xffffffffu, in ? rbs : (1 << 20)));
            rMax = max(rMax, __reduce_max_sync(0xffffffffu, in ? rbs : -1));
            // ---- deposit, sample after sample (fixed order); lanes 0..15 own the 16 (node, corner) products
            if (lane < 16) {
                const int off = dep_off + (m & (kTcGroup - 1)) * SN + (1 - gB0) * S;
                const double* pw = wb + (v >> 2) * kTcPitch;
                const double* pc = cc + (v & 3) * kTcPitch;
                for (int s = pos; s < pend; ++s) Wt[off + base[s]] += pw[s] * pc[s];
            }
            __syncwarp();
            pos = pend;
        }
        k += nb;
    }
    if (have) flush();
}

}  // namespace e2e
