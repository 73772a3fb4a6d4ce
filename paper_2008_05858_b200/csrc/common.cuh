// common.cuh -- shared declarations of libe2e (device views of the handles, error plumbing).
// CUDA path only: nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>
#include <atomic>
#include <string>
#include <vector>
#include <mutex>
#include <memory>

#include "../../include/e2e.h"

namespace e2e {

// ------------------------------------------------------------------------------------------------
// limits
// ------------------------------------------------------------------------------------------------
constexpr int kMaxDeg = 5;
constexpr int kMaxCoef = (kMaxDeg + 1) * (kMaxDeg + 1);
constexpr int kMaxFibers = 64;     // spectra travel as a kernel parameter
constexpr int kMaxTerms = 32;      // chord-quadrature terms (node pairs): Q <= 64
constexpr int kBinShift = 6;       // 64-column bins of the per-order row-range summary
constexpr int kBinPad = 256;       // bins cover x in [-kBinPad, nx + kBinPad)

// ------------------------------------------------------------------------------------------------
// error plumbing
// ------------------------------------------------------------------------------------------------
void set_error(const std::string& msg);
int fail(int code, const std::string& msg);
int fail_cuda(cudaError_t e, const char* what);
extern std::atomic<long long> g_launches;
inline void count_launch(int n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }

#define E2E_CUDA(call)                                                   \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return ::e2e::fail_cuda(e__, #call);     \
    } while (0)

// ------------------------------------------------------------------------------------------------
// O2 / G8: spectral-format polynomial, fma-Horner in the fixed order
//   inner over q = deg_m..0 in M, outer over p = deg_l..0 in L, every step acc = fma(acc, var, coef).
// P:63 "centroid coordinates" of each spectral fiber image.  Bit-identical on host and device (IEEE fma).
// ------------------------------------------------------------------------------------------------
__host__ __device__ inline double poly2(const double* c, int deg_l, int deg_m, double L, double M)
{
    double acc = 0.0;
    for (int p = deg_l; p >= 0; --p) {
        double inner = 0.0;
        for (int q = deg_m; q >= 0; --q) inner = fma(inner, M, c[p * (deg_m + 1) + q]);
        acc = fma(acc, L, inner);
    }
    return acc;
}

// device view of a format handle; travels by value as a kernel parameter
struct FormatView {
    int nx, ny, n_orders, n_fibers, deg_l, deg_m;
    double lam0, inv_dlam, m0, inv_dm;
    double coef_x[kMaxCoef], coef_y[kMaxCoef];
    const int* order_m;            // [n_orders]
    const double* lam_min;         // [n_orders]
    const double* dl;              // [n_orders] wavelength step of the order's sample grid
    const long long* nsamp;        // [n_orders]
    const double* blaze_lam_c;     // [n_orders]
    const double* blaze_amp;       // [n_orders] or nullptr
    const double* fiber_dx;        // [n_fibers]
    const double* fiber_dy;
    const double* inner_x;         // [n_orders][kMaxDeg + 1] inner Horner sums over M of coef_x, zero-padded at the top
    const double* inner_y;         //   (O2: the order number is constant along a strip, so these are the per-order
                                   //    coefficients of the outer Horner in L; same fma sequence -> same bits)
    const double* eff_table;       // or nullptr
    long long eff_n;
    double eff_lam0, eff_dlam;
};

struct SpectraParam {
    e2e_spectrum_t s[kMaxFibers];
};

// one (fiber, order) strip of consecutive samples inside the workspace arrays
struct Strip {
    long long off;   // first sample in x/y/w
    long long n;     // sample count
};

// work item of the render kernels: a run of consecutive 32-sample chunks of one strip
struct Item {
    int strip;
    int chunk0;
    int nchunks;
};

// analytic PSF (O4): chord-quadrature terms after pairing the nodes +-s
struct AnalyticParam {
    int n_terms;
    int by_gauss;                  // 1: y-factor is the plain pixel-integrated gaussian (Dy = 0)
    double inv_sx, inv_sy;         // 1/sigma
    double hbx, hby;               // footprint half-width + 1/2 (G9)
    double s[kMaxTerms];           // chord abscissa a cos(theta) >= 0, in px
    double cs[kMaxTerms];          // chord half-length over sigma_y
    double wq[kMaxTerms];          // quadrature weight (2/(Q+1)) sin^2(theta)
    double g[kMaxTerms];           // sigma_y / (2 c): scale of the y-factor (1 when by_gauss)
    unsigned paired;               // bit t: term t stands for the two nodes +-s[t]
};

// analytic PSF, production path: pixel-phase polynomial tables (poly_tables.h, render_poly.cuh)
struct PolyParam {
    int T;                             // chord terms
    int nlo_x, ncol, ncol_pad;         // window columns X + nlo_x + [0, ncol)
    int nlo_y, nrow, nrow_pad;
    double hbx, hby;                   // footprint half-width + 1/2 (G9)
    const double* tx;                  // [T][P+1][ncol_pad]
    const double* ty;                  // [T][P+1][nrow_pad]
};

// analytic PSF, dense sampling: footprint-cell moments (poly_tables.h MomentTables, render_moment.cuh)
struct MomentParam {
    int T;                             // chord terms
    int ncol, nrow;                    // largest footprint in columns / rows
    int nit, njt;                      // 8-wide tiles per axis
    double hbx, hby;                   // footprint half-width + 1/2 (G9)
    double c0x, c0y;                   // phase origin: d = (x - ilo) - c0x
    const double2* fx;                 // [T][nit][npt][32] fragment-ordered coefficient pairs
    const double2* fy;                 // [nyb][T][njt][32]   y-phase windows, degree 7 (one power tile)
    int nyb;                           // windows: centres -1/2 + (b + 1/2)/nyb, valid for |dy - centre| <= 1/nyb
    // analytic PSF map (G21): gx x gy nodes, node n's tables at fx + n * fx_node_stride, fy + n * fy_node_stride (0 x 0: one PSF)
    int gx, gy;
    double fsx, fsy;                   // (gx-1)/(nx-1), (gy-1)/(ny-1)
    size_t fx_node_stride, fy_node_stride;
};

struct TabParam {
    int npix, os, n;               // n = npix * os cells per axis
    int gx, gy;
    int ld;                        // leading dimension of one summed-area table (n + 1)
    double hb;                     // npix/2 + 1/2
    double half;                   // npix / 2
    double fsx, fsy;               // (gx-1)/(nx-1), (gy-1)/(ny-1)
    const double* sat;             // [gy][gx][n+1][n+1] summed-area tables
    const double* pi;              // [gy][gx][os][os][pi_ld][pi_ld] phase-major pixel-integral tables (render_tabcell.cuh) or nullptr
    int pi_ld;                     // npix + 2
    double c0;                     // hb - 1: sub-pixel phase = (x - ilo) - c0 in (0, 1]
};

}  // namespace e2e

// handles ------------------------------------------------------------------------------------------
struct e2e_psf {
    int kind;
    int nx, ny;
    double hbx, hby;
    int fp_cols, fp_rows;          // largest footprint in columns / rows
    int Q;
    e2e::AnalyticParam an;
    e2e::TabParam tab;
    double* d_sat = nullptr;
    double* d_pi = nullptr;        // phase-major pixel-integral tables of the tabulated PSF
    int poly_degree = 0;           // > 0: polynomial tables built (analytic PSF), degree in use
    double poly_trunc_err = 0.0;   // measured truncation error of the tables
    e2e::PolyParam poly;
    double* d_poly = nullptr;      // one allocation: tx then ty
    int moment_npt = 0;            // > 0: moment tables built, power tiles in use
    int moment_degree = 0;         // x-phase degree of the moment tables
    e2e::MomentParam mom;
    double* d_mom = nullptr;       // one allocation: fx then fy
    bool is_map = false;           // analytic PSF map (G21): mom holds one table set per node
    ~e2e_psf();                    // frees the device tables (also on the early returns of e2e_psf_create)
};

struct e2e_plan {                  // schedule for one (format, footprint) pair; cached in the format handle
    double hbx, hby;
    int nyb = 0;                   // y-phase windows of the PSF's moment tables the cell ranges below were counted for (0: none)
    long long n_cells = 0;         // footprint cells of the whole frame
    long long* d_cell_off = nullptr;   // [n_items + 1] first cell of every item (two-kernel render, render_cells.cuh)
    int win_cols, win_rows;        // window capacity the schedule was built for
    int n_strips = 0;
    long long total_samples = 0;
    std::vector<e2e::Strip> strips;
    e2e::Strip* d_strips = nullptr;
    int n_phases = 0;
    std::vector<int> phase_off;    // [n_phases + 1] into d_items
    e2e::Item* d_items = nullptr;
    int n_items = 0;
    int n_colors = 0;
    bool small = false;            // a frame whose items cannot fill the GPU (K > 2 run classes): wide CTAs render its items
    // dependency lists of the persistent render launch (render_moment.cuh): item i waits for dep_idx[dep_off[i] .. dep_off[i+1])
    // -- every item earlier in the queue (= lower index) whose pixels may overlap its own
    int* d_dep_off = nullptr;
    int* d_dep_idx = nullptr;
    std::vector<int> dep_off, dep_idx;
    int* d_succ_off = nullptr;         // the transposed lists: the items that wait for item i
    int* d_succ_idx = nullptr;
    unsigned* d_ctrl_init = nullptr;   // initial control block: head counters 0, then the number of dependencies per item
    // The same items regrouped into row bands that share no pixel (build_plan).  `host`: up to 8 bands of growing size for
    // e2e_render_frame_host (finished rows travel to the host while later bands render); `halves`: 2 equal bands that
    // e2e_render_frame renders concurrently on two streams (the tail of one band's launch overlaps the other band's work).
    // phase_off[b * (n_phases_all + 1) + ph] indexes d_items; rows below fin_row[b] belong to bands <= b only.
    struct BandPart {
        int n_bands = 0;
        std::vector<int> phase_off, fin_row, strip_off;
        e2e::Item* d_items = nullptr;
        int* d_strips = nullptr;
        std::vector<int> queue_off;    // [n_bands + 1] into d_queue: the band's item ids in queue order (persistent launch)
        int* d_queue = nullptr;
        std::vector<double> lam_lo, lam_hi;   // [n_bands][n_fibers] wavelength range of the band's samples of one fiber (lo > hi: none)
    };
    BandPart host, halves, host16;     // host16: fewer, equal bands for the host path's uint16 output (short copies)
    int n_phases_all = 0;          // phases before empty ones were dropped (colour x class)
    // streams and events the library adds to the caller's stream (second compute stream, copy stream of the host path): owned by
    // the plan, so renders of different (format, psf) pairs never wait on each other's forked work; created on first use
    void* pipe = nullptr;
    std::mutex pipe_mu;
    ~e2e_plan();
};

struct e2e_format {
    e2e::FormatView view;          // device pointers inside
    std::vector<int> order_m;
    std::vector<double> lam_min, lam_max, dl, fiber_dx, fiber_dy;
    std::vector<long long> nsamp;
    std::vector<double> min_spacing;   // [n_orders] smallest |x_{k+1} - x_k|
    std::vector<double> bin_ymin, bin_ymax;   // [n_orders][n_bins] base-trace row range per 64-column bin
    int n_bins = 0;
    long long samples_per_fiber = 0;
    double samples_per_px = 0;
    void* d_blob = nullptr;        // one device allocation holding every per-order array
    std::mutex plan_mu;
    std::vector<std::unique_ptr<e2e_plan>> plans;
};
