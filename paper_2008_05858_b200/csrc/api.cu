// api.cu -- the C ABI of include/e2e.h: handle creation / validation, the host-side schedule, kernel launches.
#include "common.cuh"
#include "setup.cuh"
#include "render_analytic.cuh"
#include "render_tabulated.cuh"
#include "render_tabcell.cuh"
#include "render_poly.cuh"
#include "render_moment.cuh"
#include "plan_check.cuh"
#include "render_cells.cuh"
#include "poly_tables.h"

#include <algorithm>
#include <cstring>
#include <cstdlib>
#include <cmath>

namespace e2e {

// ------------------------------------------------------------------------------------------------
// error plumbing
// ------------------------------------------------------------------------------------------------
static thread_local std::string t_error;
std::atomic<long long> g_launches{0};

void set_error(const std::string& msg) { t_error = msg; }
int fail(int code, const std::string& msg) { t_error = msg; return code; }
int fail_cuda(cudaError_t e, const char* what)
{
    t_error = std::string(what) + ": " + cudaGetErrorString(e);
    return E2E_ERR_CUDA;
}

int launch_detector(const double* d_in, double* d_out, long long n, const e2e_detector_t& det, cudaStream_t stream, long long p0 = 0);
int launch_detector_ex(const double* d_in, void* d_out, bool out16, long long n, int nx, const e2e_detector_ex_t& det,
                       cudaStream_t stream, long long p0 = 0);
int measure_fp64_peak(int repeats, double* burst, double* sustained);
int probe_fp64_pipe(double* r);

// samples per pixel from which the per-cell moment kernel beats the per-sample polynomial kernel
constexpr double kMomentMinSpp = 8.0;
constexpr long long kSmallFrameItems = 4736;   // 2 x (148 SMs x 16 resident warps): below this a K = 2 schedule leaves the GPU idle
#ifndef E2E_SPLIT
#define E2E_SPLIT 1                    // 1: e2e_render_frame renders the analytic PSF with the two kernels of render_cells.cuh
#endif
constexpr int kDeviceParts = 2;        // row bands e2e_render_frame renders concurrently (they share no pixel)
#ifndef E2E_HOST_BANDS
#define E2E_HOST_BANDS 8
#endif
#ifndef E2E_HOST_BANDS16
#define E2E_HOST_BANDS16 5
#endif
constexpr int kHostBands = E2E_HOST_BANDS;       // row bands of e2e_render_frame_host (device-to-host copy overlapped with rendering)
constexpr int kHostBands16 = E2E_HOST_BANDS16;   // the same for the uint16 output: the copy is 4x shorter, fewer and larger bands pay

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------------------------------------
// per-stage device timing (e2e_profile_*): event pairs recorded on the caller's stream, resolved on read
// ------------------------------------------------------------------------------------------------
enum Stage { kStageZero = 0, kStageSetup, kStageRender, kStageDetector, kNumStages };
struct Pending { int stage; cudaEvent_t a, b; };
static std::mutex g_prof_mu;
static bool g_prof_on = false;
static std::vector<Pending> g_prof_pending;
static std::vector<cudaEvent_t> g_prof_free;
static e2e_profile_t g_prof_tot = {};

static cudaEvent_t prof_event()
{
    if (!g_prof_free.empty()) { cudaEvent_t e = g_prof_free.back(); g_prof_free.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
// RAII bracket of one stage; inert while profiling is off
struct StageTimer {
    cudaStream_t stream; int stage; cudaEvent_t a = nullptr; bool on;
    StageTimer(int stage_, cudaStream_t s) : stream(s), stage(stage_)
    {
        std::lock_guard<std::mutex> lk(g_prof_mu);
        on = g_prof_on;
        if (on) { a = prof_event(); if (a) cudaEventRecord(a, stream); else on = false; }
    }
    ~StageTimer()
    {
        if (!on) return;
        std::lock_guard<std::mutex> lk(g_prof_mu);
        cudaEvent_t b = prof_event();
        if (!b) { g_prof_free.push_back(a); return; }
        cudaEventRecord(b, stream);
        g_prof_pending.push_back(Pending{stage, a, b});
    }
};
static inline bool is_fin(double v) { return std::isfinite(v); }

// host copy of sample_position's x (same operation sequence: O1, O2)
static double host_x_of_lambda(const e2e_format_desc_t& d, int o, double lam)
{
    double L = (lam - d.lam0) * d.inv_dlam;
    double M = ((double)d.order_m[o] - d.m0) * d.inv_dm;
    return poly2(d.coef_x, d.deg_l, d.deg_m, L, M);
}

}  // namespace e2e

using namespace e2e;

// second compute stream, copy stream and events of one plan (fork / join around the caller's stream); created on first use
struct HostPipe {
    static constexpr int kEvents = 16;
    cudaStream_t copy = nullptr;
    cudaStream_t up = nullptr;         // host -> device: the spectrum tables travel in the order the bands need them
    cudaStream_t aux = nullptr;        // second compute stream: odd bands render here while even bands render on the caller's
    cudaEvent_t ev[kEvents] = {};
    cudaEvent_t ev_up[kEvents] = {};
    cudaEvent_t ev_start = nullptr, ev_aux_done = nullptr, ev_zero = nullptr;
    std::mutex mu;                     // one call at a time enqueues on these streams
    ~HostPipe()
    {
        if (copy) cudaStreamDestroy(copy);
        if (up) cudaStreamDestroy(up);
        if (aux) cudaStreamDestroy(aux);
        for (cudaEvent_t e : ev)
            if (e) cudaEventDestroy(e);
        for (cudaEvent_t e : ev_up)
            if (e) cudaEventDestroy(e);
        if (ev_start) cudaEventDestroy(ev_start);
        if (ev_aux_done) cudaEventDestroy(ev_aux_done);
        if (ev_zero) cudaEventDestroy(ev_zero);
    }
};
static HostPipe* host_pipe(e2e_plan* pl)
{
    std::lock_guard<std::mutex> lk(pl->pipe_mu);
    if (!pl->pipe) {
        HostPipe* h = new HostPipe;
        bool ok = cudaStreamCreateWithFlags(&h->copy, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaStreamCreateWithFlags(&h->up, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaStreamCreateWithFlags(&h->aux, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaEventCreateWithFlags(&h->ev_start, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&h->ev_aux_done, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&h->ev_zero, cudaEventDisableTiming) == cudaSuccess;
        for (int i = 0; ok && i < HostPipe::kEvents; ++i)
            ok = cudaEventCreateWithFlags(&h->ev[i], cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&h->ev_up[i], cudaEventDisableTiming) == cudaSuccess;
        if (!ok) { delete h; return nullptr; }
        pl->pipe = h;
    }
    return static_cast<HostPipe*>(pl->pipe);
}

e2e_psf::~e2e_psf()
{
    if (d_sat) cudaFree(d_sat);
    if (d_pi) cudaFree(d_pi);
    if (d_poly) cudaFree(d_poly);
    if (d_mom) cudaFree(d_mom);
}

e2e_plan::~e2e_plan()
{
    delete static_cast<HostPipe*>(pipe);
    if (d_strips) cudaFree(d_strips);
    if (d_items) cudaFree(d_items);
    if (d_dep_off) cudaFree(d_dep_off);
    if (d_dep_idx) cudaFree(d_dep_idx);
    if (d_succ_off) cudaFree(d_succ_off);
    if (d_succ_idx) cudaFree(d_succ_idx);
    if (d_ctrl_init) cudaFree(d_ctrl_init);
    if (d_cell_off) cudaFree(d_cell_off);
    for (BandPart* bp : {&host, &halves, &host16}) {
        if (bp->d_items) cudaFree(bp->d_items);
        if (bp->d_strips) cudaFree(bp->d_strips);
        if (bp->d_queue) cudaFree(bp->d_queue);
    }
}

extern "C" {

const char* e2e_last_error(void) { return t_error.c_str(); }
const char* e2e_version(void) { return "e2e-b200 0.1 sm_100a"; }
int64_t e2e_launch_count(void) { return (int64_t)g_launches.load(); }

// ================================================================================================
// format
// ================================================================================================
int e2e_format_create(e2e_format_t** out, const e2e_format_desc_t* d)
{
    if (!out) return fail(E2E_ERR_INVALID_ARG, "format_create: out is NULL");
    *out = nullptr;
    if (!d) return fail(E2E_ERR_INVALID_ARG, "format_create: desc is NULL");
    if (d->nx <= 0 || d->ny <= 0 || d->nx > (1 << 20) || d->ny > (1 << 20))
        return fail(E2E_ERR_INVALID_ARG, "format_create: bad detector size");
    if (d->n_orders <= 0 || d->n_orders > 4096) return fail(E2E_ERR_INVALID_ARG, "format_create: n_orders out of range");
    if (d->n_fibers <= 0) return fail(E2E_ERR_INVALID_ARG, "format_create: n_fibers must be >= 1");
    if (d->n_fibers > kMaxFibers) return fail(E2E_ERR_UNSUPPORTED, "format_create: more than 64 fibers");
    if (d->deg_l < 0 || d->deg_l > kMaxDeg || d->deg_m < 0 || d->deg_m > kMaxDeg)
        return fail(E2E_ERR_INVALID_ARG, "format_create: polynomial degree must be 0..5");
    if (!d->order_m || !d->lam_min || !d->lam_max || !d->fiber_dx || !d->fiber_dy || !d->coef_x || !d->coef_y ||
        !d->blaze_lam_c)
        return fail(E2E_ERR_INVALID_ARG, "format_create: NULL array");
    if (!(d->samples_per_px > 0.0) || !is_fin(d->samples_per_px))
        return fail(E2E_ERR_INVALID_ARG, "format_create: samples_per_px must be > 0");
    if (!is_fin(d->lam0) || !is_fin(d->inv_dlam) || !is_fin(d->m0) || !is_fin(d->inv_dm))
        return fail(E2E_ERR_INVALID_ARG, "format_create: non-finite normalisation");
    const int nc = (d->deg_l + 1) * (d->deg_m + 1);
    for (int i = 0; i < nc; ++i)
        if (!is_fin(d->coef_x[i]) || !is_fin(d->coef_y[i])) return fail(E2E_ERR_INVALID_ARG, "format_create: non-finite coefficient");
    for (int o = 0; o < d->n_orders; ++o) {
        if (!is_fin(d->lam_min[o]) || !is_fin(d->lam_max[o]) || !(d->lam_min[o] < d->lam_max[o]))
            return fail(E2E_ERR_INVALID_ARG, "format_create: need lam_min < lam_max for every order");
        if (!is_fin(d->blaze_lam_c[o]) || (d->blaze_amp && !is_fin(d->blaze_amp[o])))
            return fail(E2E_ERR_INVALID_ARG, "format_create: non-finite blaze parameter");
    }
    for (int f = 0; f < d->n_fibers; ++f)
        if (!is_fin(d->fiber_dx[f]) || !is_fin(d->fiber_dy[f])) return fail(E2E_ERR_INVALID_ARG, "format_create: non-finite fiber offset");
    if (d->eff_table && (d->eff_n < 2 || !(d->eff_dlam > 0.0) || !is_fin(d->eff_lam0)))
        return fail(E2E_ERR_INVALID_ARG, "format_create: bad efficiency table");

    std::unique_ptr<e2e_format> F(new (std::nothrow) e2e_format);
    if (!F) return fail(E2E_ERR_NOMEM, "format_create: out of host memory");
    const int no = d->n_orders, nf = d->n_fibers;
    F->order_m.assign(d->order_m, d->order_m + no);
    F->lam_min.assign(d->lam_min, d->lam_min + no);
    F->lam_max.assign(d->lam_max, d->lam_max + no);
    F->fiber_dx.assign(d->fiber_dx, d->fiber_dx + nf);
    F->fiber_dy.assign(d->fiber_dy, d->fiber_dy + nf);
    F->samples_per_px = d->samples_per_px;
    F->dl.resize(no);
    F->nsamp.resize(no);
    long long total = 0, nmax = 0;
    for (int o = 0; o < no; ++o) {
        // a1: N_m = ceil(spp * |x(lam_max) - x(lam_min)|)
        double xa = host_x_of_lambda(*d, o, d->lam_min[o]), xb = host_x_of_lambda(*d, o, d->lam_max[o]);
        double n = std::ceil(d->samples_per_px * std::fabs(xb - xa));
        if (!(n >= 0.0)) n = 0.0;
        if (n > 2.0e9) return fail(E2E_ERR_UNSUPPORTED, "format_create: more than 2e9 samples in one order");
        F->nsamp[o] = (long long)n;
        F->dl[o] = n > 0.0 ? (d->lam_max[o] - d->lam_min[o]) / n : 0.0;
        total += F->nsamp[o];
        nmax = std::max(nmax, F->nsamp[o]);
    }
    F->samples_per_fiber = total;

    // one device blob with every per-order / per-fiber array
    size_t off = 0;
    auto reserve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_m = reserve(sizeof(int) * no), o_lmin = reserve(8 * no), o_dl = reserve(8 * no), o_ns = reserve(8 * no);
    const size_t o_bl = reserve(8 * no), o_ba = reserve(8 * no), o_fx = reserve(8 * nf), o_fy = reserve(8 * nf);
    const size_t o_ix = reserve(8 * (size_t)no * (kMaxDeg + 1)), o_iy = reserve(8 * (size_t)no * (kMaxDeg + 1));
    const size_t o_eff = reserve(d->eff_table ? 8 * (size_t)d->eff_n : 0);
    char* blob = nullptr;
    E2E_CUDA(cudaMalloc(&blob, off));
    F->d_blob = blob;
    auto fail_free = [&](int code) { cudaFree(blob); F->d_blob = nullptr; return code; };
#define E2E_CUDA_F(call)                                                         \
    do {                                                                         \
        cudaError_t e__ = (call);                                                \
        if (e__ != cudaSuccess) return fail_free(fail_cuda(e__, #call));         \
    } while (0)
    E2E_CUDA_F(cudaMemcpy(blob + o_m, d->order_m, sizeof(int) * no, cudaMemcpyHostToDevice));
    E2E_CUDA_F(cudaMemcpy(blob + o_lmin, d->lam_min, 8 * no, cudaMemcpyHostToDevice));
    E2E_CUDA_F(cudaMemcpy(blob + o_dl, F->dl.data(), 8 * no, cudaMemcpyHostToDevice));
    E2E_CUDA_F(cudaMemcpy(blob + o_ns, F->nsamp.data(), 8 * no, cudaMemcpyHostToDevice));
    E2E_CUDA_F(cudaMemcpy(blob + o_bl, d->blaze_lam_c, 8 * no, cudaMemcpyHostToDevice));
    if (d->blaze_amp) E2E_CUDA_F(cudaMemcpy(blob + o_ba, d->blaze_amp, 8 * no, cudaMemcpyHostToDevice));
    E2E_CUDA_F(cudaMemcpy(blob + o_fx, d->fiber_dx, 8 * nf, cudaMemcpyHostToDevice));
    E2E_CUDA_F(cudaMemcpy(blob + o_fy, d->fiber_dy, 8 * nf, cudaMemcpyHostToDevice));
    {
        // O2 inner Horner sums over M per order (the exact fma sequence of poly2's inner loop), zero-padded to degree 5
        std::vector<double> ix((size_t)no * (kMaxDeg + 1), 0.0), iy((size_t)no * (kMaxDeg + 1), 0.0);
        for (int o = 0; o < no; ++o) {
            const double M = ((double)d->order_m[o] - d->m0) * d->inv_dm;
            for (int p = 0; p <= d->deg_l; ++p) {
                double sx = 0.0, sy = 0.0;
                for (int q = d->deg_m; q >= 0; --q) {
                    sx = fma(sx, M, d->coef_x[p * (d->deg_m + 1) + q]);
                    sy = fma(sy, M, d->coef_y[p * (d->deg_m + 1) + q]);
                }
                ix[(size_t)o * (kMaxDeg + 1) + p] = sx;
                iy[(size_t)o * (kMaxDeg + 1) + p] = sy;
            }
        }
        E2E_CUDA_F(cudaMemcpy(blob + o_ix, ix.data(), 8 * ix.size(), cudaMemcpyHostToDevice));
        E2E_CUDA_F(cudaMemcpy(blob + o_iy, iy.data(), 8 * iy.size(), cudaMemcpyHostToDevice));
    }
    if (d->eff_table) E2E_CUDA_F(cudaMemcpy(blob + o_eff, d->eff_table, 8 * (size_t)d->eff_n, cudaMemcpyHostToDevice));

    FormatView& v = F->view;
    memset(&v, 0, sizeof(v));
    v.nx = d->nx; v.ny = d->ny; v.n_orders = no; v.n_fibers = nf; v.deg_l = d->deg_l; v.deg_m = d->deg_m;
    v.lam0 = d->lam0; v.inv_dlam = d->inv_dlam; v.m0 = d->m0; v.inv_dm = d->inv_dm;
    for (int i = 0; i < nc; ++i) { v.coef_x[i] = d->coef_x[i]; v.coef_y[i] = d->coef_y[i]; }
    v.order_m = (const int*)(blob + o_m);
    v.lam_min = (const double*)(blob + o_lmin);
    v.dl = (const double*)(blob + o_dl);
    v.nsamp = (const long long*)(blob + o_ns);
    v.blaze_lam_c = (const double*)(blob + o_bl);
    v.blaze_amp = d->blaze_amp ? (const double*)(blob + o_ba) : nullptr;
    v.fiber_dx = (const double*)(blob + o_fx);
    v.fiber_dy = (const double*)(blob + o_fy);
    v.inner_x = (const double*)(blob + o_ix);
    v.inner_y = (const double*)(blob + o_iy);
    v.eff_table = d->eff_table ? (const double*)(blob + o_eff) : nullptr;
    v.eff_n = d->eff_n; v.eff_lam0 = d->eff_lam0; v.eff_dlam = d->eff_dlam;

    // device pass over every sample: monotonicity, spacing, row range per 64-column bin
    const int n_bins = (d->nx + 2 * kBinPad + (1 << kBinShift) - 1) >> kBinShift;
    F->n_bins = n_bins;
    const size_t nb = (size_t)no * n_bins;
    unsigned long long* scratch = nullptr;
    E2E_CUDA_F(cudaMalloc(&scratch, 8 * (2 * (size_t)no + 2 * nb)));
    unsigned long long *d_smin = scratch, *d_smax = scratch + no, *d_ymin = scratch + 2 * no, *d_ymax = d_ymin + nb;
    cudaMemset(d_smin, 0xff, 8 * (size_t)no);
    cudaMemset(d_smax, 0x00, 8 * (size_t)no);
    cudaMemset(d_ymin, 0xff, 8 * nb);
    cudaMemset(d_ymax, 0x00, 8 * nb);
    if (nmax > 0) {
        dim3 grid((unsigned)((nmax + 255) / 256), (unsigned)no);
        scan_format_kernel<<<grid, 256>>>(v, n_bins, d_smin, d_smax, d_ymin, d_ymax);
        count_launch();
    }
    std::vector<unsigned long long> h(2 * (size_t)no + 2 * nb);
    cudaError_t ce = cudaMemcpy(h.data(), scratch, 8 * h.size(), cudaMemcpyDeviceToHost);
    cudaFree(scratch);
    if (ce != cudaSuccess) return fail_free(fail_cuda(ce, "format_create: scan"));
    F->min_spacing.assign(no, 0.0);
    F->bin_ymin.assign(nb, INFINITY);
    F->bin_ymax.assign(nb, -INFINITY);
    std::vector<double> max_spacing(no, 0.0);
    for (int o = 0; o < no; ++o) {
        if (F->nsamp[o] >= 2) {
            if (h[o] == ~0ULL || h[no + o] == 0ULL) return fail_free(fail(E2E_ERR_CUDA, "format_create: scan produced no spacing"));
            double dmin = dec_double(h[o]), dmax = dec_double(h[no + o]);
            if (!(dmin > 0.0) && !(dmax < 0.0)) {
                char buf[160];
                snprintf(buf, sizeof buf, "format_create: x(lambda) is not strictly monotone in order index %d (m=%d)", o, d->order_m[o]);
                return fail_free(fail(E2E_ERR_NOT_MONOTONIC, buf));
            }
            F->min_spacing[o] = std::min(std::fabs(dmin), std::fabs(dmax));
            max_spacing[o] = std::max(std::fabs(dmin), std::fabs(dmax));
        }
        for (int b = 0; b < n_bins; ++b) {
            unsigned long long a = h[2 * (size_t)no + (size_t)o * n_bins + b], c = h[2 * (size_t)no + nb + (size_t)o * n_bins + b];
            if (a != ~0ULL && c != 0ULL) {
                F->bin_ymin[(size_t)o * n_bins + b] = dec_double(a);
                F->bin_ymax[(size_t)o * n_bins + b] = dec_double(c);
            }
        }
    }
    // keep max spacing behind min spacing (same vector, second half) to avoid another member
    F->min_spacing.insert(F->min_spacing.end(), max_spacing.begin(), max_spacing.end());
#undef E2E_CUDA_F
    *out = F.release();
    return E2E_OK;
}

void e2e_format_destroy(e2e_format_t* fmt)
{
    if (!fmt) return;
    fmt->plans.clear();
    if (fmt->d_blob) cudaFree(fmt->d_blob);
    delete fmt;
}

int e2e_format_num_samples(const e2e_format_t* fmt, int64_t* n_per_order, int64_t* n_total)
{
    if (!fmt) return fail(E2E_ERR_INVALID_ARG, "format_num_samples: fmt is NULL");
    if (n_per_order)
        for (size_t o = 0; o < fmt->nsamp.size(); ++o) n_per_order[o] = fmt->nsamp[o];
    if (n_total) *n_total = fmt->samples_per_fiber * fmt->view.n_fibers;
    return E2E_OK;
}

// ================================================================================================
// psf
// ================================================================================================
// Q chosen so that the Gauss-Chebyshev chord quadrature is converged below 1e-12 of the PSF peak:
// measured against Q = 64 for D/(2 sigma) in [0, 3.3]
static int auto_nodes(double a, double b, double sx, double sy)
{
    double r = std::max(a / sx, b / sy);
    int q = (int)std::ceil(7.0 + 3.0 * r);
    q += q & 1;
    return std::min(std::max(q, 8), 64);
}

int e2e_psf_create(e2e_psf_t** out, const e2e_psf_desc_t* d, int32_t nx, int32_t ny)
{
    if (!out) return fail(E2E_ERR_INVALID_ARG, "psf_create: out is NULL");
    *out = nullptr;
    if (!d) return fail(E2E_ERR_INVALID_ARG, "psf_create: desc is NULL");
    if (nx <= 0 || ny <= 0) return fail(E2E_ERR_INVALID_ARG, "psf_create: bad detector size");
    std::unique_ptr<e2e_psf> P(new (std::nothrow) e2e_psf);
    if (!P) return fail(E2E_ERR_NOMEM, "psf_create: out of host memory");
    memset(&P->an, 0, sizeof(P->an));
    memset(&P->tab, 0, sizeof(P->tab));
    memset(&P->poly, 0, sizeof(P->poly));
    memset(&P->mom, 0, sizeof(P->mom));
    P->kind = d->kind; P->nx = nx; P->ny = ny; P->Q = 0;
    if (d->kind == 0) {
        const bool is_map = d->an_sigma_x != nullptr || d->an_sigma_y != nullptr;
        int n_map = 1;
        if (is_map) {
            if (!d->an_sigma_x || !d->an_sigma_y || d->an_gx < 1 || d->an_gy < 1)
                return fail(E2E_ERR_INVALID_ARG, "psf_create: bad analytic PSF map description");
            if ((long long)d->an_gx * d->an_gy > 64) return fail(E2E_ERR_UNSUPPORTED, "psf_create: more than 64 nodes in the analytic PSF map");
            n_map = d->an_gx * d->an_gy;
            for (int c = 0; c < n_map; ++c)
                if (!(d->an_sigma_x[c] > 0.0) || !(d->an_sigma_y[c] > 0.0) || !is_fin(d->an_sigma_x[c]) || !is_fin(d->an_sigma_y[c]))
                    return fail(E2E_ERR_INVALID_ARG, "psf_create: sigma must be > 0 at every node");
        } else if (!(d->sigma_x > 0.0) || !(d->sigma_y > 0.0) || !is_fin(d->sigma_x) || !is_fin(d->sigma_y))
            return fail(E2E_ERR_INVALID_ARG, "psf_create: sigma must be > 0");
        if (!(d->fiber_dx_px >= 0.0) || !(d->fiber_dy_px >= 0.0) || !is_fin(d->fiber_dx_px) || !is_fin(d->fiber_dy_px))
            return fail(E2E_ERR_INVALID_ARG, "psf_create: fiber widths must be >= 0");
        if (!is_fin(d->support_nsigma)) return fail(E2E_ERR_INVALID_ARG, "psf_create: support_nsigma not finite");
        if (d->n_nodes < 0) return fail(E2E_ERR_INVALID_ARG, "psf_create: n_nodes < 0");
        if (d->n_nodes > 2 * kMaxTerms) return fail(E2E_ERR_UNSUPPORTED, "psf_create: n_nodes > 64");
        const double t = d->support_nsigma > 0.0 ? d->support_nsigma : 7.5;
        const double a = 0.5 * d->fiber_dx_px, b = 0.5 * d->fiber_dy_px;
        // G9: H = D/2 + t sigma; footprint = all pixels touching [x - H, x + H].  G21: ONE box from the largest node sigma
        double sx_box = d->sigma_x, sy_box = d->sigma_y, sx_min = d->sigma_x, sy_min = d->sigma_y;
        if (is_map) {
            sx_box = sx_min = d->an_sigma_x[0]; sy_box = sy_min = d->an_sigma_y[0];
            for (int c = 1; c < n_map; ++c) {
                sx_box = std::max(sx_box, d->an_sigma_x[c]); sy_box = std::max(sy_box, d->an_sigma_y[c]);
                sx_min = std::min(sx_min, d->an_sigma_x[c]); sy_min = std::min(sy_min, d->an_sigma_y[c]);
            }
        }
        const double Hx = 0.5 * d->fiber_dx_px + t * sx_box, Hy = 0.5 * d->fiber_dy_px + t * sy_box;
        P->hbx = Hx + 0.5; P->hby = Hy + 0.5;
        if (2.0 * P->hbx + 1.0 > 96.0 || 2.0 * P->hby + 1.0 > 96.0)
            return fail(E2E_ERR_UNSUPPORTED, "psf_create: footprint larger than 96 px");
        // chord terms of one (sigma_x, sigma_y): nodes q and Q+1-q share |s|, c and the weight -> one term with
        // F(d) = Phi(d - s) + Phi(d + s).  Q = the caller's, else chosen for the narrowest sigma of the map
        const bool pure_gauss = !(a > 0.0) && !(b > 0.0);
        const int Qn = pure_gauss ? 1 : (d->n_nodes > 0 ? d->n_nodes : auto_nodes(a, b, sx_min, sy_min));
        P->Q = Qn;
        auto chord_terms = [&](double sy, AnalyticParam& A) {
            A.by_gauss = !(b > 0.0);
            A.paired = 0;
            if (pure_gauss) {                     // P2: pure gaussian, one term
                A.n_terms = 1; A.s[0] = 0.0; A.cs[0] = 0.0; A.wq[0] = 1.0; A.g[0] = 1.0;
                return;
            }
            int nt = 0;
            for (int q = 1; 2 * q <= Qn + 1; ++q) {
                const long double th = (long double)q * 3.14159265358979323846264338327950288L / (long double)(Qn + 1);
                const long double sn = sinl(th), cn = cosl(th);
                A.s[nt] = (double)((long double)a * cn);
                const long double c = (long double)b * sn;
                A.cs[nt] = (double)(c / (long double)sy);
                A.wq[nt] = (double)((2.0L / (long double)(Qn + 1)) * sn * sn);
                A.g[nt] = b > 0.0 ? (double)((long double)sy / (2.0L * c)) : 1.0;
                if (2 * q != Qn + 1) A.paired |= 1u << nt;
                else A.s[nt] = 0.0;               // middle node of an odd rule sits at s = 0
                ++nt;
            }
            A.n_terms = nt;
        };
        auto shape_of = [&](double sx, double sy, const AnalyticParam& A) {
            PsfShape shape;
            shape.sx = sx; shape.sy = sy; shape.by_gauss = A.by_gauss != 0;
            for (int i = 0; i < A.n_terms; ++i) {
                ChordTerm ct;
                ct.s = A.s[i]; ct.cs = A.cs[i]; ct.wq = A.wq[i]; ct.g = A.g[i]; ct.paired = (A.paired >> i) & 1u;
                shape.terms.push_back(ct);
            }
            return shape;
        };
        AnalyticParam& A = P->an;
        A.inv_sx = 1.0 / sx_box; A.inv_sy = 1.0 / sy_box;
        A.hbx = P->hbx; A.hby = P->hby;
        chord_terms(is_map ? sy_box : d->sigma_y, A);
        if (is_map) {
            // analytic PSF map: one moment-table set per node, all with the same layout (x degree, y windows) = the
            // finest any node needs.  No per-sample-polynomial or direct fallback: the map needs the cell-moment kernel.
            P->is_map = true;
            std::vector<MomentTables> tabs(n_map);
            std::vector<AnalyticParam> An(n_map);
            int Pmax = 0, nybmax = 0;
            for (int c = 0; c < n_map; ++c) {
                memset(&An[c], 0, sizeof(AnalyticParam));
                chord_terms(d->an_sigma_y[c], An[c]);
                if (!build_moment_tables(shape_of(d->an_sigma_x[c], d->an_sigma_y[c], An[c]), P->hbx, P->hby, tabs[c]))
                    return fail(E2E_ERR_UNSUPPORTED, "psf_create: no converged moment tables for a node of the PSF map (sigma too small)");
                Pmax = std::max(Pmax, tabs[c].P); nybmax = std::max(nybmax, tabs[c].nyb);
            }
            for (int c = 0; c < n_map; ++c)
                if (tabs[c].P != Pmax || tabs[c].nyb != nybmax) {
                    tabs[c] = MomentTables();
                    if (!build_moment_tables(shape_of(d->an_sigma_x[c], d->an_sigma_y[c], An[c]), P->hbx, P->hby, tabs[c], Pmax, nybmax))
                        return fail(E2E_ERR_UNSUPPORTED, "psf_create: PSF map nodes do not share a table layout");
                }
            if (tabs[0].npt > 4) return fail(E2E_ERR_UNSUPPORTED, "psf_create: PSF map needs an x degree above 31");
            const size_t nfx = tabs[0].fx.size(), nfy = tabs[0].fy.size();
            for (int c = 1; c < n_map; ++c)
                if (tabs[c].fx.size() != nfx || tabs[c].fy.size() != nfy) return fail(E2E_ERR_UNSUPPORTED, "psf_create: PSF map table sizes differ");
            E2E_CUDA(cudaMalloc(&P->d_mom, 8 * (nfx + nfy) * (size_t)n_map));
            cudaError_t ce = cudaSuccess;
            for (int c = 0; c < n_map && ce == cudaSuccess; ++c) {
                ce = cudaMemcpy(P->d_mom + nfx * c, tabs[c].fx.data(), 8 * nfx, cudaMemcpyHostToDevice);
                if (ce == cudaSuccess) ce = cudaMemcpy(P->d_mom + nfx * n_map + nfy * c, tabs[c].fy.data(), 8 * nfy, cudaMemcpyHostToDevice);
            }
            if (ce != cudaSuccess) { cudaFree(P->d_mom); P->d_mom = nullptr; return fail_cuda(ce, "psf_create: PSF map table upload"); }
            const MomentTables& mom = tabs[0];
            MomentParam& M = P->mom;
            M.T = mom.T; M.ncol = mom.ncol; M.nrow = mom.nrow; M.nit = mom.nit; M.njt = mom.njt;
            M.hbx = P->hbx; M.hby = P->hby; M.c0x = mom.c0x; M.c0y = mom.c0y; M.nyb = mom.nyb;
            M.fx = reinterpret_cast<const double2*>(P->d_mom);
            M.fy = reinterpret_cast<const double2*>(P->d_mom + nfx * n_map);
            M.gx = d->an_gx; M.gy = d->an_gy;
            M.fsx = nx > 1 ? (double)(d->an_gx - 1) / (double)(nx - 1) : 0.0;
            M.fsy = ny > 1 ? (double)(d->an_gy - 1) / (double)(ny - 1) : 0.0;
            M.fx_node_stride = nfx / 2; M.fy_node_stride = nfy / 2;
            P->moment_npt = mom.npt;
            P->moment_degree = mom.P;
        } else {
            // production path: pixel-phase polynomial tables (the direct special-function kernel stays as the fallback
            // for PSFs whose tables do not converge: sigma below ~0.3 px)
            const PsfShape shape = shape_of(d->sigma_x, d->sigma_y, A);
            A.inv_sx = 1.0 / d->sigma_x; A.inv_sy = 1.0 / d->sigma_y;
            PolyTables tabs;
            if (build_poly_tables(shape, P->hbx, P->hby, tabs) && tabs.ncol_pad <= kMaxWin && tabs.nrow_pad <= kMaxWin) {
                const size_t nx_ = tabs.tx.size(), ny_ = tabs.ty.size();
                E2E_CUDA(cudaMalloc(&P->d_poly, 8 * (nx_ + ny_)));
                cudaError_t ce = cudaMemcpy(P->d_poly, tabs.tx.data(), 8 * nx_, cudaMemcpyHostToDevice);
                if (ce == cudaSuccess) ce = cudaMemcpy(P->d_poly + nx_, tabs.ty.data(), 8 * ny_, cudaMemcpyHostToDevice);
                if (ce != cudaSuccess) { cudaFree(P->d_poly); P->d_poly = nullptr; return fail_cuda(ce, "psf_create: polynomial table upload"); }
                PolyParam& Q = P->poly;
                Q.T = tabs.T; Q.nlo_x = tabs.nlo_x; Q.ncol = tabs.ncol; Q.ncol_pad = tabs.ncol_pad;
                Q.nlo_y = tabs.nlo_y; Q.nrow = tabs.nrow; Q.nrow_pad = tabs.nrow_pad;
                Q.hbx = P->hbx; Q.hby = P->hby; Q.tx = P->d_poly; Q.ty = P->d_poly + nx_;
                P->poly_degree = tabs.P;
                P->poly_trunc_err = (double)tabs.trunc_err;
            }
            // dense sampling: footprint-cell moment tables (render_moment.cuh)
            MomentTables mom;
            if (P->poly_degree > 0 && build_moment_tables(shape, P->hbx, P->hby, mom) && mom.npt <= 4) {
                const size_t nfx = mom.fx.size(), nfy = mom.fy.size();
                E2E_CUDA(cudaMalloc(&P->d_mom, 8 * (nfx + nfy)));
                cudaError_t ce = cudaMemcpy(P->d_mom, mom.fx.data(), 8 * nfx, cudaMemcpyHostToDevice);
                if (ce == cudaSuccess) ce = cudaMemcpy(P->d_mom + nfx, mom.fy.data(), 8 * nfy, cudaMemcpyHostToDevice);
                if (ce != cudaSuccess) { cudaFree(P->d_mom); P->d_mom = nullptr; return fail_cuda(ce, "psf_create: moment table upload"); }
                MomentParam& M = P->mom;
                M.T = mom.T; M.ncol = mom.ncol; M.nrow = mom.nrow; M.nit = mom.nit; M.njt = mom.njt;
                M.hbx = P->hbx; M.hby = P->hby; M.c0x = mom.c0x; M.c0y = mom.c0y; M.nyb = mom.nyb;
                M.fx = reinterpret_cast<const double2*>(P->d_mom);
                M.fy = reinterpret_cast<const double2*>(P->d_mom + nfx);
                P->moment_npt = mom.npt;
                P->moment_degree = mom.P;
            }
        }
    } else if (d->kind == 1) {
        if (d->tab_npix < 1 || d->tab_os < 1 || d->tab_gx < 1 || d->tab_gy < 1 || !d->tab)
            return fail(E2E_ERR_INVALID_ARG, "psf_create: bad tabulated PSF description");
        const long long n = (long long)d->tab_npix * d->tab_os;
        if (n > 256 || d->tab_npix > 94) return fail(E2E_ERR_UNSUPPORTED, "psf_create: tabulated kernel larger than 256 cells / 94 px");
        if ((long long)d->tab_gx * d->tab_gy > 4096) return fail(E2E_ERR_UNSUPPORTED, "psf_create: more than 4096 field nodes");
        const size_t ncell = (size_t)n * n, nk = (size_t)d->tab_gx * d->tab_gy;
        for (size_t i = 0; i < ncell * nk; ++i)
            if (!is_fin(d->tab[i])) return fail(E2E_ERR_INVALID_ARG, "psf_create: non-finite table value");
        P->hbx = P->hby = 0.5 * (double)d->tab_npix + 0.5;
        TabParam& T = P->tab;
        T.npix = d->tab_npix; T.os = d->tab_os; T.n = (int)n; T.gx = d->tab_gx; T.gy = d->tab_gy; T.ld = (int)n + 1;
        T.hb = P->hbx; T.half = 0.5 * (double)d->tab_npix;
        T.fsx = nx > 1 ? (double)(d->tab_gx - 1) / (double)(nx - 1) : 0.0;
        T.fsy = ny > 1 ? (double)(d->tab_gy - 1) / (double)(ny - 1) : 0.0;
        // T2: summed-area table C[b][a] = sum of cells [0,b) x [0,a), accumulated in long double
        const size_t ld = (size_t)n + 1;
        std::vector<double> sat(nk * ld * ld, 0.0);
        std::vector<long double> rowacc(ld);
        for (size_t k = 0; k < nk; ++k) {
            const double* Tk = d->tab + k * ncell;
            double* S = sat.data() + k * ld * ld;
            std::fill(rowacc.begin(), rowacc.end(), 0.0L);
            for (size_t bb = 1; bb <= (size_t)n; ++bb) {
                long double run = 0.0L;
                for (size_t aa = 1; aa <= (size_t)n; ++aa) {
                    run += (long double)Tk[(bb - 1) * n + (aa - 1)];
                    rowacc[aa] += run;
                    S[bb * ld + aa] = (double)rowacc[aa];
                }
            }
        }
        E2E_CUDA(cudaMalloc(&P->d_sat, 8 * sat.size()));
        cudaError_t ce = cudaMemcpy(P->d_sat, sat.data(), 8 * sat.size(), cudaMemcpyHostToDevice);
        if (ce != cudaSuccess) { cudaFree(P->d_sat); P->d_sat = nullptr; return fail_cuda(ce, "psf_create: table upload"); }
        T.sat = P->d_sat;
        // production path (render_tabcell.cuh): PI[ry][rx][J][I] = sum of the kernel cells inside the pixel whose
        // lower-left corner is the fine-grid point (os I + rx - os, os J + ry - os), from a long double SAT
        T.pi = nullptr; T.pi_ld = d->tab_npix + 2; T.c0 = P->hbx - 1.0;
        if (d->tab_os <= kTcMaxOs) {
            const int os = d->tab_os, pld = T.pi_ld, N = (int)n;
            const size_t per_node = (size_t)os * os * pld * pld;
            std::vector<double> pi(nk * per_node, 0.0);
            std::vector<long double> L(ld * ld);
            auto clampi = [&](int g) { return g < 0 ? 0 : (g > N ? N : g); };
            for (size_t k = 0; k < nk; ++k) {
                const double* Tk = d->tab + k * ncell;
                std::fill(L.begin(), L.end(), 0.0L);
                for (size_t bb = 1; bb <= (size_t)N; ++bb) {
                    long double run = 0.0L;
                    for (size_t aa = 1; aa <= (size_t)N; ++aa) {
                        run += (long double)Tk[(bb - 1) * N + (aa - 1)];
                        L[bb * ld + aa] = L[(bb - 1) * ld + aa] + run;
                    }
                }
                double* out = pi.data() + k * per_node;
                for (int ry = 0; ry < os; ++ry)
                    for (int rx = 0; rx < os; ++rx)
                        for (int J = 0; J < pld; ++J)
                            for (int I = 0; I < pld; ++I) {
                                const int gy0 = clampi(os * J + ry - os), gy1 = clampi(os * J + ry);
                                const int gx0 = clampi(os * I + rx - os), gx1 = clampi(os * I + rx);
                                const long double v = (L[(size_t)gy1 * ld + gx1] - L[(size_t)gy0 * ld + gx1]) -
                                                      (L[(size_t)gy1 * ld + gx0] - L[(size_t)gy0 * ld + gx0]);
                                out[(((size_t)ry * os + rx) * pld + J) * pld + I] = (double)v;
                            }
            }
            E2E_CUDA(cudaMalloc(&P->d_pi, 8 * pi.size()));
            ce = cudaMemcpy(P->d_pi, pi.data(), 8 * pi.size(), cudaMemcpyHostToDevice);
            if (ce != cudaSuccess) { cudaFree(P->d_pi); P->d_pi = nullptr; return fail_cuda(ce, "psf_create: pixel-integral table upload"); }
            T.pi = P->d_pi;
        }
    } else {
        return fail(E2E_ERR_INVALID_ARG, "psf_create: kind must be 0 or 1");
    }
    P->fp_cols = (int)std::floor(2.0 * P->hbx) + 1;
    P->fp_rows = (int)std::floor(2.0 * P->hby) + 1;
    *out = P.release();
    return E2E_OK;
}

int e2e_psf_info(const e2e_psf_t* psf, int32_t* n_nodes, int32_t* footprint_cols, int32_t* footprint_rows)
{
    if (!psf) return fail(E2E_ERR_INVALID_ARG, "psf_info: psf is NULL");
    if (n_nodes) *n_nodes = psf->Q;
    if (footprint_cols) *footprint_cols = psf->fp_cols;
    if (footprint_rows) *footprint_rows = psf->fp_rows;
    return E2E_OK;
}

void e2e_psf_destroy(e2e_psf_t* psf) { delete psf; }      // ~e2e_psf frees the device tables

}  // extern "C"

// ================================================================================================
// schedule: strips, runs, colours, phases
// ================================================================================================
namespace e2e {

struct Interval { int lo, hi, strip; };

static int build_plan(e2e_format* F, const e2e_psf* P, e2e_plan** out)
{
    std::lock_guard<std::mutex> lock(F->plan_mu);
    // the cell ranges of the two-kernel render depend on the y-phase windows of the PSF's tables as well
    const int nyb_key = (P->kind == 0 && P->moment_npt > 0 && !P->is_map) ? P->mom.nyb : 0;
    for (auto& p : F->plans)
        if (p->hbx == P->hbx && p->hby == P->hby && p->nyb == nyb_key) { *out = p.get(); return E2E_OK; }
    std::unique_ptr<e2e_plan> pl(new e2e_plan);
    pl->hbx = P->hbx; pl->hby = P->hby; pl->nyb = nyb_key;
    const int no = F->view.n_orders, nf = F->view.n_fibers, nx = F->view.nx;
    const int n_strips = no * nf;
    if (n_strips > 65535) return fail(E2E_ERR_UNSUPPORTED, "render: more than 65535 (fiber, order) strips");
    pl->n_strips = n_strips;
    pl->strips.resize(n_strips);
    long long off = 0;
    for (int f = 0; f < nf; ++f)
        for (int o = 0; o < no; ++o) {
            pl->strips[f * no + o] = Strip{off, F->nsamp[o]};
            off += F->nsamp[o];
        }
    pl->total_samples = off;
    const double* min_sp = F->min_spacing.data();
    const double* max_sp = F->min_spacing.data() + no;

    // ---- colours: strips whose pixel coverage may overlap must not run in the same launch
    const int nB = (nx + 63) >> 6;
    std::vector<int> cov_lo((size_t)n_strips * nB, 1), cov_hi((size_t)n_strips * nB, 0);   // empty: lo > hi
    for (int f = 0; f < nf; ++f)
        for (int o = 0; o < no; ++o) {
            if (F->nsamp[o] == 0) continue;
            const int s = f * no + o;
            const double margin = P->hbx + 2.0 + 32.0 * max_sp[o];
            if (margin + std::fabs(F->fiber_dx[f]) > (double)kBinPad)
                return fail(E2E_ERR_UNSUPPORTED, "render: footprint + fiber offset + 32 sample spacings exceeds 256 px");
            for (int B = 0; B < nB; ++B) {
                const double lo = 64.0 * B - margin - F->fiber_dx[f], hi = 64.0 * B + 63.0 + margin - F->fiber_dx[f];
                int b0 = (int)std::floor((lo + kBinPad) / 64.0), b1 = (int)std::floor((hi + kBinPad) / 64.0);
                b0 = std::max(b0, 0); b1 = std::min(b1, F->n_bins - 1);
                double ymin = INFINITY, ymax = -INFINITY;
                for (int b = b0; b <= b1; ++b) {
                    ymin = std::min(ymin, F->bin_ymin[(size_t)o * F->n_bins + b]);
                    ymax = std::max(ymax, F->bin_ymax[(size_t)o * F->n_bins + b]);
                }
                if (!(ymin <= ymax)) continue;
                double rlo = std::floor(ymin + F->fiber_dy[f] - P->hby) - 1.0, rhi = std::ceil(ymax + F->fiber_dy[f] + P->hby) + 1.0;
                rlo = std::max(rlo, -1.0e9); rhi = std::min(rhi, 1.0e9);
                cov_lo[(size_t)s * nB + B] = (int)rlo;
                cov_hi[(size_t)s * nB + B] = (int)rhi;
            }
        }
    std::vector<std::vector<int>> adj(n_strips);
    std::vector<Interval> iv;
    for (int B = 0; B < nB; ++B) {
        iv.clear();
        for (int s = 0; s < n_strips; ++s)
            if (cov_lo[(size_t)s * nB + B] <= cov_hi[(size_t)s * nB + B])
                iv.push_back(Interval{cov_lo[(size_t)s * nB + B], cov_hi[(size_t)s * nB + B], s});
        std::sort(iv.begin(), iv.end(), [](const Interval& a, const Interval& b) { return a.lo < b.lo || (a.lo == b.lo && a.strip < b.strip); });
        for (size_t i = 0; i < iv.size(); ++i)
            for (size_t j = i + 1; j < iv.size() && iv[j].lo <= iv[i].hi; ++j) {
                adj[iv[i].strip].push_back(iv[j].strip);
                adj[iv[j].strip].push_back(iv[i].strip);
            }
    }
    std::vector<int> color(n_strips, -1);
    int n_colors = 0;
    std::vector<char> used;
    for (int s = 0; s < n_strips; ++s) {
        used.assign(n_colors + 1, 0);
        for (int t : adj[s])
            if (color[t] >= 0) used[color[t]] = 1;
        int c = 0;
        while (used[c]) ++c;
        color[s] = c;
        n_colors = std::max(n_colors, c + 1);
    }
    pl->n_colors = n_colors;

    // ---- runs: consecutive runs of a strip cycle through K launches; two runs of the same class are separated by
    //      K - 1 full runs whose joint x-extent exceeds 2 hb + 3 px, so their pixel windows are disjoint.
    //      K = 2 (long runs, fewest launches) when that already fills the GPU; small frames (a single strip) take
    //      K = 4: runs 3x shorter, twice the launches, 4/3 G chunk-times per strip end to end instead of 2 G
    //      (measured on B200, tiny / rv_sweep render: K = 2 0.49 / 0.95 ms, K = 4 0.40 / 0.68, K = 8 0.42 / 0.70, K = 16 0.54 / 0.77)
    auto run_length = [&](int o, long long nchunks) {
        long long G = nchunks;
        const long long N = F->nsamp[o];
        if (N >= 2 && min_sp[o] > 0.0) {
            double g = std::floor((2.0 * P->hbx + 3.0) / (32.0 * min_sp[o])) + 1.0;
            if (g < (double)nchunks) G = (long long)g;
        }
        return G;
    };
    long long items_k2 = 0;
    for (int s = 0; s < n_strips; ++s) {
        const long long N = F->nsamp[s % no];
        if (N == 0) continue;
        const long long nchunks = (N + 31) / 32;
        items_k2 += (nchunks + run_length(s % no, nchunks) - 1) / run_length(s % no, nchunks);
    }
#ifndef E2E_SMALL_K
#define E2E_SMALL_K 8
#endif
    const int K = items_k2 < kSmallFrameItems ? ((P->kind == 0 && P->moment_npt > 0) ? E2E_SMALL_K : 4) : 2;
    pl->small = K > 2;
    std::vector<std::vector<Item>> phases((size_t)n_colors * K);
    for (int s = 0; s < n_strips; ++s) {
        const int o = s % no;
        const long long N = F->nsamp[o];
        if (N == 0) continue;
        const long long nchunks = (N + 31) / 32;
        long long G = run_length(o, nchunks);
        if (K > 2 && G < nchunks) G = (G + K - 2) / (K - 1);
        // runs are kept at the minimum length: twice as long measured 4.39 against 4.48 ms for the device-resident flush launch
        // (fewer cells cut at item ends), but the host path's per-band launches then have too few items to fill the GPU
        // (e2e 15.3 against 13.9 ms fp64, 9.9 against 8.1 ms uint16)
        int run = 0;
        for (long long c0 = 0; c0 < nchunks; c0 += G, ++run)
            phases[(size_t)color[s] * K + (run % K)].push_back(Item{s, (int)c0, (int)std::min(G, nchunks - c0)});
    }
    std::vector<Item> flat;
    pl->phase_off.clear();
    pl->phase_off.push_back(0);
    for (auto& ph : phases) {
        if (ph.empty()) continue;
        flat.insert(flat.end(), ph.begin(), ph.end());
        pl->phase_off.push_back((int)flat.size());
    }
    pl->n_phases = (int)pl->phase_off.size() - 1;
    pl->n_items = (int)flat.size();
    // ---- dependency lists for the persistent launch (render_moment.cuh).  The queue order is the order of `flat`
    //      (phase-major); item i depends on every item j < i that may share a pixel with it: same strip or a strip whose
    //      rows may overlap (adj, from the per-bin row coverage above), and overlapping column ranges.  Column range of an
    //      item = footprint boxes of its first and last sample (x is monotone along a strip).
    {
        const FormatView& v = F->view;
        auto host_x = [&](int o, long long k) {
            const double lam = fma((double)k + 0.5, F->dl[o], F->lam_min[o]);
            const double L = (lam - v.lam0) * v.inv_dlam, M = ((double)F->order_m[o] - v.m0) * v.inv_dm;
            return poly2(v.coef_x, v.deg_l, v.deg_m, L, M);
        };
        const int ni = (int)flat.size();
        std::vector<int> clo(ni), chi(ni);
        struct Run { int clo, chi, idx; };
        std::vector<std::vector<Run>> runs(n_strips);
        for (int i = 0; i < ni; ++i) {
            const Item& it = flat[i];
            const int f = it.strip / no, o = it.strip % no;
            const long long k0 = (long long)it.chunk0 * 32;
            const long long k1 = std::min<long long>(F->nsamp[o], ((long long)it.chunk0 + it.nchunks) * 32) - 1;
            const double xa = host_x(o, k0) + F->fiber_dx[f], xb = host_x(o, k1) + F->fiber_dx[f];
            // exactly the first column of the leftmost box and the last column of the rightmost one (G9: ceil(x - hbx),
            // floor(x + hbx); host_x runs the device's operation sequence, so these are the device's integers).  No padding:
            // a padded range would link runs of one class to each other and serialise the strip (e2e_plan_check verifies
            // on the device that no edge is missing)
            const double lo = std::max(std::min(xa, xb) - P->hbx, -1.0e9), hi = std::min(std::max(xa, xb) + P->hbx, 1.0e9);
            clo[i] = (int)std::ceil(lo); chi[i] = (int)std::floor(hi);
            runs[it.strip].push_back(Run{clo[i], chi[i], i});
        }
        for (auto& r : runs) std::sort(r.begin(), r.end(), [](const Run& a, const Run& b) { return a.clo < b.clo || (a.clo == b.clo && a.idx < b.idx); });
        for (auto& a : adj) { std::sort(a.begin(), a.end()); a.erase(std::unique(a.begin(), a.end()), a.end()); }
        pl->dep_off.assign(ni + 1, 0);
        pl->dep_idx.clear();
        std::vector<int> mine;
        for (int i = 0; i < ni; ++i) {
            const int s = flat[i].strip;
            mine.clear();
            auto scan = [&](int t) {
                const std::vector<Run>& r = runs[t];
                // runs are consecutive along x: clo and chi both ascend; first run with chi >= clo[i]
                size_t lo = 0, hi = r.size();
                while (lo < hi) { const size_t mid = (lo + hi) / 2; if (r[mid].chi < clo[i]) lo = mid + 1; else hi = mid; }
                // chi is not strictly sorted when a strip ends with a short run: step back over equal / larger values
                while (lo > 0 && r[lo - 1].chi >= clo[i]) --lo;
                for (size_t j = lo; j < r.size() && r[j].clo <= chi[i]; ++j)
                    if (r[j].chi >= clo[i] && r[j].idx < i) mine.push_back(r[j].idx);
            };
            scan(s);
            for (int t : adj[s]) scan(t);
            std::sort(mine.begin(), mine.end());
            pl->dep_idx.insert(pl->dep_idx.end(), mine.begin(), mine.end());
            pl->dep_off[i + 1] = (int)pl->dep_idx.size();
        }
        // transposed lists (successors) and the initial control block
        {
            std::vector<int> soff(ni + 1, 0), sidx(pl->dep_idx.size());
            for (int j : pl->dep_idx) soff[j + 1] += 1;
            for (int i = 0; i < ni; ++i) soff[i + 1] += soff[i];
            std::vector<int> fill(soff.begin(), soff.end() - 1);
            for (int i = 0; i < ni; ++i)
                for (int d = pl->dep_off[i]; d < pl->dep_off[i + 1]; ++d) sidx[fill[pl->dep_idx[d]]++] = i;
            std::vector<unsigned> init((size_t)kCtrlHeads + std::max(ni, 1), 0u);
            for (int i = 0; i < ni; ++i) init[kCtrlHeads + i] = (unsigned)(pl->dep_off[i + 1] - pl->dep_off[i]);
            E2E_CUDA(cudaMalloc(&pl->d_succ_off, sizeof(int) * (ni + 1)));
            E2E_CUDA(cudaMemcpy(pl->d_succ_off, soff.data(), sizeof(int) * (ni + 1), cudaMemcpyHostToDevice));
            E2E_CUDA(cudaMalloc(&pl->d_succ_idx, sizeof(int) * std::max<size_t>(1, sidx.size())));
            if (!sidx.empty()) E2E_CUDA(cudaMemcpy(pl->d_succ_idx, sidx.data(), sizeof(int) * sidx.size(), cudaMemcpyHostToDevice));
            E2E_CUDA(cudaMalloc(&pl->d_ctrl_init, sizeof(unsigned) * init.size()));
            E2E_CUDA(cudaMemcpy(pl->d_ctrl_init, init.data(), sizeof(unsigned) * init.size(), cudaMemcpyHostToDevice));
        }
        E2E_CUDA(cudaMalloc(&pl->d_dep_off, sizeof(int) * (ni + 1)));
        E2E_CUDA(cudaMemcpy(pl->d_dep_off, pl->dep_off.data(), sizeof(int) * (ni + 1), cudaMemcpyHostToDevice));
        E2E_CUDA(cudaMalloc(&pl->d_dep_idx, sizeof(int) * std::max<size_t>(1, pl->dep_idx.size())));
        if (!pl->dep_idx.empty())
            E2E_CUDA(cudaMemcpy(pl->d_dep_idx, pl->dep_idx.data(), sizeof(int) * pl->dep_idx.size(), cudaMemcpyHostToDevice));
    }
    E2E_CUDA(cudaMalloc(&pl->d_strips, sizeof(Strip) * std::max(1, n_strips)));
    E2E_CUDA(cudaMemcpy(pl->d_strips, pl->strips.data(), sizeof(Strip) * n_strips, cudaMemcpyHostToDevice));
    E2E_CUDA(cudaMalloc(&pl->d_items, sizeof(Item) * std::max<size_t>(1, flat.size())));
    if (!flat.empty()) E2E_CUDA(cudaMemcpy(pl->d_items, flat.data(), sizeof(Item) * flat.size(), cudaMemcpyHostToDevice));
    // ---- cells of every item (two-kernel render): the render's own cell walk, positions straight from the format
    if (nyb_key > 0 && !flat.empty()) {
        const int ni = (int)flat.size();
        int* d_counts = nullptr;
        E2E_CUDA(cudaMalloc(&d_counts, sizeof(int) * ni));
        CellStore none;
        memset(&none, 0, sizeof(none));
        static SpectraParam no_spectra;
        const unsigned blocks = (unsigned)((ni + kCellWarps - 1) / kCellWarps);
        switch (P->moment_npt) {
            case 2: cell_moment_kernel<2, true, false><<<blocks, kCellWarps * 32>>>(nullptr, nullptr, nullptr, pl->d_strips, pl->d_items, nullptr, ni, P->mom, none, d_counts, F->view, no_spectra, nullptr, 0, nullptr); break;
            case 3: cell_moment_kernel<3, true, false><<<blocks, kCellWarps * 32>>>(nullptr, nullptr, nullptr, pl->d_strips, pl->d_items, nullptr, ni, P->mom, none, d_counts, F->view, no_spectra, nullptr, 0, nullptr); break;
            default: cell_moment_kernel<4, true, false><<<blocks, kCellWarps * 32>>>(nullptr, nullptr, nullptr, pl->d_strips, pl->d_items, nullptr, ni, P->mom, none, d_counts, F->view, no_spectra, nullptr, 0, nullptr); break;
        }
        count_launch();
        std::vector<int> counts(ni);
        cudaError_t ce = cudaMemcpy(counts.data(), d_counts, sizeof(int) * ni, cudaMemcpyDeviceToHost);
        cudaFree(d_counts);
        if (ce != cudaSuccess) return fail_cuda(ce, "render: cell count");
        std::vector<long long> off(ni + 1, 0);
        for (int i = 0; i < ni; ++i) off[i + 1] = off[i] + counts[i];
        pl->n_cells = off[ni];
        E2E_CUDA(cudaMalloc(&pl->d_cell_off, sizeof(long long) * (ni + 1)));
        E2E_CUDA(cudaMemcpy(pl->d_cell_off, off.data(), sizeof(long long) * (ni + 1), cudaMemcpyHostToDevice));
    }
    // ---- row bands: strips sorted by their first row, split into bands by sample count, bands starting only at gaps
    {
        const int ny = F->view.ny;
        std::vector<int> rlo(n_strips, INT_MAX), rhi(n_strips, INT_MIN);
        for (int s = 0; s < n_strips; ++s)
            for (int B = 0; B < nB; ++B)
                if (cov_lo[(size_t)s * nB + B] <= cov_hi[(size_t)s * nB + B]) {
                    rlo[s] = std::min(rlo[s], cov_lo[(size_t)s * nB + B]);
                    rhi[s] = std::max(rhi[s], cov_hi[(size_t)s * nB + B]);
                }
        std::vector<int> order(n_strips);
        for (int s = 0; s < n_strips; ++s) order[s] = s;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return rlo[a] < rlo[b]; });
        pl->n_phases_all = (int)phases.size();
        const long long tot = std::max<long long>(pl->total_samples, 1);
        auto build_part = [&](int want, bool ramp, e2e_plan::BandPart& part) -> int {
            // band b takes the share wgt[b] of the samples; ramp: the first bands are small, so that the copy engine starts
            // early, the later ones up to 3x larger (the copy is the slower side and must only never run dry)
            std::vector<double> cum(want + 1, 0.0);
            {
                std::vector<double> wgt(want, 1.0);
                if (ramp)
                    for (int b = 0; b < want; ++b) wgt[b] = 1.0 + 2.0 * (double)b / (double)std::max(1, want - 1);
                double sum = 0.0;
                for (double w : wgt) sum += w;
                for (int b = 0; b < want; ++b) cum[b + 1] = cum[b] + wgt[b] / sum;
            }
            // A band may only start at a GAP -- a strip whose first row lies above every row of the strips before it -- so
            // that no pixel belongs to two bands: bands can be rendered concurrently (two streams) and the rows of a band
            // are final as soon as that band alone is done.  Without enough gaps (orders that overlap everywhere) there are
            // fewer bands, down to one.
            std::vector<int> band_of(n_strips, 0);
            long long acc = 0;
            int cur_band = 0, top = INT_MIN;
            for (int i = 0; i < n_strips; ++i) {
                const int s = order[i];
                if (pl->strips[s].n == 0) { band_of[s] = cur_band; continue; }
                const double frac = (double)acc / (double)tot;
                int b = 0;
                while (b < want - 1 && frac >= cum[b + 1]) ++b;
                if (b > cur_band && rlo[s] > top) cur_band = std::min(b, cur_band + 1);
                band_of[s] = cur_band;
                top = std::max(top, rhi[s]);
                acc += pl->strips[s].n;
            }
            want = cur_band + 1;
            part.n_bands = want;
            part.fin_row.assign(want, ny);
            for (int b = want - 2; b >= 0; --b) {
                int lo = part.fin_row[b + 1];
                for (int s = 0; s < n_strips; ++s)
                    if (band_of[s] == b + 1 && pl->strips[s].n > 0) lo = std::min(lo, rlo[s]);
                part.fin_row[b] = std::max(0, std::min(lo, ny));
            }
            std::vector<Item> bflat;
            part.phase_off.assign((size_t)want * (phases.size() + 1), 0);
            for (int b = 0; b < want; ++b)
                for (size_t ph = 0; ph <= phases.size(); ++ph) {
                    part.phase_off[(size_t)b * (phases.size() + 1) + ph] = (int)bflat.size();
                    if (ph == phases.size()) break;
                    for (const Item& it : phases[ph])
                        if (band_of[it.strip] == b) bflat.push_back(it);
                }
            std::vector<int> bstrips;
            part.strip_off.assign(want + 1, 0);
            for (int b = 0; b < want; ++b) {
                for (int s = 0; s < n_strips; ++s)
                    if (band_of[s] == b && pl->strips[s].n > 0) bstrips.push_back(s);
                part.strip_off[b + 1] = (int)bstrips.size();
            }
            // wavelength range each band reads from each fiber's spectrum (the host path uploads the tables in that order)
            const int nf = F->view.n_fibers, no = F->view.n_orders;
            part.lam_lo.assign((size_t)want * nf, INFINITY);
            part.lam_hi.assign((size_t)want * nf, -INFINITY);
            for (int s = 0; s < n_strips; ++s) {
                if (pl->strips[s].n == 0) continue;
                const int fiber = s / no, o = s - fiber * no;
                double& lo = part.lam_lo[(size_t)band_of[s] * nf + fiber];
                double& hi = part.lam_hi[(size_t)band_of[s] * nf + fiber];
                lo = std::min(lo, std::min(F->lam_min[o], F->lam_max[o]));
                hi = std::max(hi, std::max(F->lam_min[o], F->lam_max[o]));
            }
            E2E_CUDA(cudaMalloc(&part.d_strips, sizeof(int) * std::max<size_t>(1, bstrips.size())));
            if (!bstrips.empty()) E2E_CUDA(cudaMemcpy(part.d_strips, bstrips.data(), sizeof(int) * bstrips.size(), cudaMemcpyHostToDevice));
            E2E_CUDA(cudaMalloc(&part.d_items, sizeof(Item) * std::max<size_t>(1, bflat.size())));
            if (!bflat.empty()) E2E_CUDA(cudaMemcpy(part.d_items, bflat.data(), sizeof(Item) * bflat.size(), cudaMemcpyHostToDevice));
            // the band's items (ids = positions in `flat`) in queue order, for the persistent launch
            std::vector<int> bq;
            part.queue_off.assign(want + 1, 0);
            for (int b = 0; b < want; ++b) {
                for (int i = 0; i < (int)flat.size(); ++i)
                    if (band_of[flat[i].strip] == b) bq.push_back(i);
                part.queue_off[b + 1] = (int)bq.size();
            }
            E2E_CUDA(cudaMalloc(&part.d_queue, sizeof(int) * std::max<size_t>(1, bq.size())));
            if (!bq.empty()) E2E_CUDA(cudaMemcpy(part.d_queue, bq.data(), sizeof(int) * bq.size(), cudaMemcpyHostToDevice));
            return E2E_OK;
        };
        // host path: 8 bands of growing size when a band's launches are few (2 colours x 2 classes); frames with many
        // colours (10 fibers per order: 10 launches per band) measured better with 6 equal bands
        const bool many_phases = phases.size() > 4;
        const int want = many_phases ? 6 : kHostBands;
        int rc = build_part(want, !many_phases, pl->host);
        if (rc) return rc;
        rc = build_part(kDeviceParts, false, pl->halves);
        if (rc) return rc;
        rc = build_part(std::min(kHostBands16, want), false, pl->host16);
        if (rc) return rc;
    }
    *out = pl.get();
    F->plans.push_back(std::move(pl));
    return E2E_OK;
}

static size_t sample_array_bytes(long long total) { return align_up((size_t)std::max<long long>(total, 1) * 8, 256); }

static int check_spectra(const e2e_format* F, const e2e_spectrum_t* spectra, const char* who)
{
    if (!spectra) return fail(E2E_ERR_INVALID_ARG, std::string(who) + ": spectra is NULL");
    for (int f = 0; f < F->view.n_fibers; ++f) {
        const e2e_spectrum_t& s = spectra[f];
        if (!s.d_flux || s.n < 2 || !(s.dlam > 0.0) || !is_fin(s.lam0) || !is_fin(s.scale) || !(s.doppler > 0.0) || !is_fin(s.doppler))
            return fail(E2E_ERR_INVALID_ARG, std::string(who) + ": bad spectrum descriptor");
    }
    return E2E_OK;
}

static int launch_setup(const e2e_format* F, const e2e_plan* pl, const e2e_spectrum_t* spectra, double* d_x, double* d_y,
                        double* d_w, cudaStream_t stream, const e2e_plan::BandPart* part = nullptr, int band = -1)
{
    SpectraParam sp;
    memset(&sp, 0, sizeof(sp));
    for (int f = 0; f < F->view.n_fibers; ++f) sp.s[f] = spectra[f];
    long long nmax = 0;
    for (long long n : F->nsamp) nmax = std::max(nmax, n);
    if (nmax == 0) return E2E_OK;
    const int* ids = nullptr;
    int ny_grid = pl->n_strips;
    if (part && band >= 0) {                                    // one row band
        ids = part->d_strips + part->strip_off[band];
        ny_grid = part->strip_off[band + 1] - part->strip_off[band];
        if (ny_grid == 0) return E2E_OK;
    }
    dim3 grid((unsigned)((nmax + 255) / 256), (unsigned)ny_grid);
    setup_samples_kernel<<<grid, 256, 0, stream>>>(F->view, sp, pl->d_strips, 0, nullptr, d_x, d_y, d_w, ids);
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "setup_samples_kernel launch");
    return E2E_OK;
}

// dense sampling -> per-cell moments; sparse sampling (few samples per footprint cell) -> per-sample polynomials
static bool choose_moment(const e2e_format* F, const e2e_psf* P)
{
    return P->kind == 0 && P->moment_npt > 0 && (F->samples_per_px >= kMomentMinSpp || P->is_map);
}

// tabulated PSF: cell-deposit kernel unless the oversampling is too fine for its weight array
static bool choose_tabcell(const e2e_psf* P) { return P->kind == 1 && P->tab.pi != nullptr; }

// control block of the persistent render launch: kCtrlHeads head counters + one flag per item (zeroed before the launch)
static size_t ctrl_bytes(const e2e_plan* pl) { return align_up(sizeof(unsigned) * ((size_t)kCtrlHeads + (size_t)std::max(pl->n_items, 1)), 256); }

// two-kernel render (render_cells.cuh): is it the path of this pair, and the bytes of its per-cell records in the workspace
static bool use_split(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl)
{
    return E2E_SPLIT != 0 && choose_moment(F, P) && !P->is_map && pl->d_cell_off != nullptr && pl->n_cells > 0;
}
static size_t cell_hdr_bytes(const e2e_plan* pl) { return align_up(sizeof(CellHeader) * (size_t)std::max<long long>(pl->n_cells, 1), 256); }
static size_t cell_mom_bytes(const e2e_plan* pl, const e2e_psf* P)
{
    return align_up(sizeof(double) * 64 * (size_t)P->moment_npt * (size_t)std::max<long long>(pl->n_cells, 1), 256);
}
static size_t cell_bytes(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl)
{
    return use_split(F, P, pl) ? cell_hdr_bytes(pl) + cell_mom_bytes(pl, P) : 0;
}

// bytes of the per-sample arrays x | y | w at the head of the workspace: none on the two-kernel path, which never materialises
// the samples
static size_t sample_arrays_bytes(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl)
{
    return use_split(F, P, pl) ? 0 : 3 * sample_array_bytes(pl->total_samples);
}

static CellStore cell_store(const e2e_plan* pl, unsigned* ctrl)
{
    CellStore cs;
    cs.cell_off = pl->d_cell_off;
    cs.hdr = (CellHeader*)((char*)ctrl + align_up(sizeof(unsigned) * ((size_t)kCtrlHeads + (size_t)std::max(pl->n_items, 1)), 256));
    cs.mom = (double*)((char*)cs.hdr + cell_hdr_bytes(pl));
    cs.frame_cells = 0;
    cs.n_frames = 1;
    return cs;
}

// kernel A of the two-kernel render: a1-a3 + the moments of every cell of the items ids[0 .. n) (nullptr: all items)
// zero_frame (16-byte aligned, even pixel count; see fused_zero_ok): the kernel also zero-fills that frame
static int launch_cell_moments(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl, const e2e_spectrum_t* spectra, unsigned* ctrl,
                               const int* ids, int n, cudaStream_t stream, double* zero_frame = nullptr)
{
    if (n <= 0) return E2E_OK;
    double2* const zero = reinterpret_cast<double2*>(zero_frame);
    const long long n_zero = zero_frame ? (long long)F->view.nx * F->view.ny / 2 : 0;
    const CellStore cs = cell_store(pl, ctrl);
    SpectraParam sp;
    memset(&sp, 0, sizeof(sp));
    for (int f = 0; f < F->view.n_fibers; ++f) sp.s[f] = spectra[f];
    const unsigned blocks = (unsigned)((n + kCellWarps - 1) / kCellWarps);
#define E2E_CELL_CASE(NPT)                                                                                                     \
    case NPT:                                                                                                                   \
        cell_moment_kernel<NPT, false, true><<<blocks, kCellWarps * 32, sizeof(MomentWarpSmem<NPT, false>) * kCellWarps, stream>>>( \
            nullptr, nullptr, nullptr, pl->d_strips, pl->d_items, ids, n, P->mom, cs, nullptr, F->view, sp, zero, n_zero, nullptr); \
        break;
    switch (P->moment_npt) {
        E2E_CELL_CASE(2) E2E_CELL_CASE(3) E2E_CELL_CASE(4)
        default: return fail(E2E_ERR_UNSUPPORTED, "render: no moment kernel for this polynomial degree");
    }
#undef E2E_CELL_CASE
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "cell_moment_kernel launch");
    return E2E_OK;
}

// kernel B: the contraction of every cell of the queue's items, in queue order
static int launch_cell_flush(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl, double* d_frame, unsigned* ctrl, const int* queue,
                             int n, int head, cudaStream_t stream)
{
    if (n <= 0) return E2E_OK;
    const CellStore cs = cell_store(pl, ctrl);
    QueueParam W;
    memset(&W, 0, sizeof(W));
    W.queue = queue; W.n = n; W.head = head; W.ctrl = ctrl;
    W.succ_off = pl->d_succ_off; W.succ_idx = pl->d_succ_idx; W.dep_off = pl->d_dep_off; W.dep_idx = pl->d_dep_idx;
    if (pl->small) {
        // a frame that cannot fill the GPU: one CTA of kWideWarps warps per item, the cell's tiles spread over the warps
        switch (P->moment_npt) {
            case 2: cell_flush_wide_kernel<2><<<(unsigned)n, kWideWarps * 32, 0, stream>>>(W, P->mom, cs, d_frame, F->view.nx, F->view.ny, nullptr); break;
            case 3: cell_flush_wide_kernel<3><<<(unsigned)n, kWideWarps * 32, 0, stream>>>(W, P->mom, cs, d_frame, F->view.nx, F->view.ny, nullptr); break;
            case 4: cell_flush_wide_kernel<4><<<(unsigned)n, kWideWarps * 32, 0, stream>>>(W, P->mom, cs, d_frame, F->view.nx, F->view.ny, nullptr); break;
            default: return fail(E2E_ERR_UNSUPPORTED, "render: no moment kernel for this polynomial degree");
        }
        count_launch();
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(e, "cell_flush_wide_kernel launch");
        return E2E_OK;
    }
    switch (P->moment_npt) {
        case 2: cell_flush_kernel<2><<<(unsigned)n, 32, 0, stream>>>(W, P->mom, cs, d_frame, F->view.nx, F->view.ny, nullptr); break;
        case 3: cell_flush_kernel<3><<<(unsigned)n, 32, 0, stream>>>(W, P->mom, cs, d_frame, F->view.nx, F->view.ny, nullptr); break;
        case 4: cell_flush_kernel<4><<<(unsigned)n, 32, 0, stream>>>(W, P->mom, cs, d_frame, F->view.nx, F->view.ny, nullptr); break;
        default: return fail(E2E_ERR_UNSUPPORTED, "render: no moment kernel for this polynomial degree");
    }
    count_launch();
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "cell_flush_kernel launch");
    return E2E_OK;
}

// (re)initialise a control block in the caller's workspace for one launch: head counters 0, dependency counters from the plan
static cudaError_t ctrl_reset(const e2e_plan* pl, unsigned* ctrl, cudaStream_t stream)
{
    return cudaMemcpyAsync(ctrl, pl->d_ctrl_init, sizeof(unsigned) * ((size_t)kCtrlHeads + (size_t)std::max(pl->n_items, 1)),
                           cudaMemcpyDeviceToDevice, stream);
}

// ---- batch form of the two-kernel render (e2e_render_frames): 1-D grids, frame = blockIdx.x % n_frames.  Workspace after the frame-pointer array:
//      SpectraParam[n_frames] | control blocks [n_frames] | cell headers [n_frames][n_cells] | moment tiles [n_frames][n_cells]
struct BatchLayout {
    size_t sp_off, ctrl_off, hdr_off, mom_off, bytes;
};
static BatchLayout batch_layout(const e2e_psf* P, const e2e_plan* pl, int n_frames, size_t ptr_bytes)
{
    BatchLayout L;
    const size_t cells = (size_t)std::max<long long>(pl->n_cells, 1) * (size_t)n_frames;
    L.sp_off = ptr_bytes;
    L.ctrl_off = L.sp_off + align_up(sizeof(SpectraParam) * (size_t)n_frames, 256);
    L.hdr_off = L.ctrl_off + ctrl_bytes(pl) * (size_t)n_frames;
    L.mom_off = L.hdr_off + align_up(sizeof(CellHeader) * cells, 256);
    L.bytes = L.mom_off + align_up(sizeof(double) * 64 * (size_t)P->moment_npt * cells, 256);
    return L;
}

static int launch_cells_batch(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl, int n_frames, const SpectraParam* d_sp,
                              unsigned* d_ctrl, const CellStore& cs, double* const* d_frames, cudaStream_t stream)
{
    const int n = pl->n_items;
    if (n <= 0) return E2E_OK;
    SpectraParam none;
    memset(&none, 0, sizeof(none));
    const long long bm = (long long)((n + kCellWarps - 1) / kCellWarps) * n_frames, bf = (long long)n * n_frames;
    if (bf > 0x7fffffffLL) return fail(E2E_ERR_UNSUPPORTED, "render_frames: more than 2^31 (item, frame) pairs");
    const unsigned gm = (unsigned)bm;
    QueueParam W;
    memset(&W, 0, sizeof(W));
    W.n = n; W.ctrl = d_ctrl; W.ctrl_stride = (long long)(ctrl_bytes(pl) / sizeof(unsigned));
    W.succ_off = pl->d_succ_off; W.succ_idx = pl->d_succ_idx; W.dep_off = pl->d_dep_off; W.dep_idx = pl->d_dep_idx;
    const unsigned gf = (unsigned)bf;
    const bool wide = pl->small;
#define E2E_BATCH_CASE(NPT)                                                                                                      \
    case NPT:                                                                                                                    \
        cell_moment_kernel<NPT, false, true, true><<<gm, kCellWarps * 32, sizeof(MomentWarpSmem<NPT, false>) * kCellWarps, stream>>>( \
            nullptr, nullptr, nullptr, pl->d_strips, pl->d_items, nullptr, n, P->mom, cs, nullptr, F->view, none, nullptr, 0, d_sp); \
        count_launch();                                                                                                          \
        if (wide) cell_flush_wide_kernel<NPT, true><<<gf, kWideWarps * 32, 0, stream>>>(W, P->mom, cs, nullptr, F->view.nx, F->view.ny, d_frames); \
        else cell_flush_kernel<NPT, true><<<gf, 32, 0, stream>>>(W, P->mom, cs, nullptr, F->view.nx, F->view.ny, d_frames);      \
        count_launch();                                                                                                          \
        break;
    switch (P->moment_npt) {
        E2E_BATCH_CASE(2) E2E_BATCH_CASE(3) E2E_BATCH_CASE(4)
        default: return fail(E2E_ERR_UNSUPPORTED, "render_frames: no moment kernel for this polynomial degree");
    }
#undef E2E_BATCH_CASE
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "render_frames: cell kernel launch");
    return E2E_OK;
}

// one queue of a persistent launch: the whole plan (queue = nullptr) or one row band of the host path
struct QueueSel {
    unsigned* ctrl = nullptr;      // zeroed control block in the caller's workspace
    const int* queue = nullptr;
    int n = 0;
    int head = 0;
};

// dynamic shared memory attribute of the moment kernel: per device, set once
template <int NPT, bool MAP>
static int moment_kernel_attr(size_t smem)
{
    static bool set[64] = {};
    int dev = 0;
    E2E_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(E2E_ERR_UNSUPPORTED, "render: device index above 63");
    if (!set[dev]) {
        E2E_CUDA(cudaFuncSetAttribute(render_moment_kernel<NPT, MAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        set[dev] = true;
    }
    return E2E_OK;
}

static int launch_render(const e2e_format* F, const e2e_psf* P, const e2e_plan* pl, const double* d_x, const double* d_y,
                         const double* d_w, double* d_frame, cudaStream_t stream, const QueueSel& qs, const Item* d_item_list = nullptr,
                         const int* phase_off = nullptr, int n_phases = -1, int n_frames = 1, long long w_stride = 0,
                         double* const* d_frames = nullptr, double* const* h_frames = nullptr)
{
    const bool use_moment = choose_moment(F, P);
    if (use_moment) {
        // production kernel: ONE launch for the whole queue, one warp per item (all frames of a batch: blockIdx.y = frame)
        if (!qs.ctrl) return fail(E2E_ERR_WORKSPACE, "render: no control block");
        if (qs.n <= 0) return E2E_OK;
        QueueParam W;
        W.queue = qs.queue; W.n = qs.n; W.dep_off = pl->d_dep_off; W.dep_idx = pl->d_dep_idx;
        W.succ_off = pl->d_succ_off; W.succ_idx = pl->d_succ_idx;
        W.ctrl = qs.ctrl; W.head = qs.head; W.ctrl_stride = (long long)(ctrl_bytes(pl) / sizeof(unsigned));
#define E2E_MOM_CASE(NPT, MAP)                                                                                          \
    case NPT: {                                                                                                         \
        const size_t sm = sizeof(MomentWarpSmem<NPT, MAP>) * kMomWarps;                                                 \
        int rc = moment_kernel_attr<NPT, MAP>(sm);                                                                      \
        if (rc) return rc;                                                                                              \
        const unsigned pb = (unsigned)((qs.n + kMomWarps - 1) / kMomWarps);                                             \
        render_moment_kernel<NPT, MAP><<<dim3(pb, n_frames), kMomWarps * 32, sm, stream>>>(                             \
            d_x, d_y, d_w, pl->d_strips, pl->d_items, W, P->mom, d_frame, F->view.nx, F->view.ny, w_stride,             \
            n_frames > 1 ? d_frames : nullptr);                                                                          \
    } break;
        if (P->is_map) {
            switch (P->moment_npt) {
                E2E_MOM_CASE(2, true) E2E_MOM_CASE(3, true) E2E_MOM_CASE(4, true)
                default: return fail(E2E_ERR_UNSUPPORTED, "render: no moment kernel for this polynomial degree");
            }
        } else {
            switch (P->moment_npt) {
                E2E_MOM_CASE(2, false) E2E_MOM_CASE(3, false) E2E_MOM_CASE(4, false)
                default: return fail(E2E_ERR_UNSUPPORTED, "render: no moment kernel for this polynomial degree");
            }
        }
#undef E2E_MOM_CASE
        count_launch();
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(e, "render_moment_kernel launch");
        return E2E_OK;
    }
    // the other kernels: one launch per phase (items of one phase share no pixel); a batch renders frame after frame
    if (n_frames > 1) {
        for (int b = 0; b < n_frames; ++b) {
            int rc = launch_render(F, P, pl, d_x, d_y, d_w + (size_t)b * w_stride, h_frames[b], stream, qs, d_item_list, phase_off, n_phases);
            if (rc) return rc;
        }
        return E2E_OK;
    }
    if (!d_item_list) { d_item_list = pl->d_items; phase_off = pl->phase_off.data(); n_phases = pl->n_phases; }
    const size_t smem_an = (size_t)kWarpsPerCta * (kWinCols + kWinRows) * kLdk * sizeof(double);
    const int lat_ld = kTabWin + 2;
    const size_t smem_tab = (size_t)kWarpsPerCta * lat_ld * lat_ld * sizeof(double);
    const bool use_tabcell = choose_tabcell(P);
    for (int ph = 0; ph < n_phases; ++ph) {
        const int i0 = phase_off[ph], n = phase_off[ph + 1] - i0;
        if (n <= 0) continue;
        const unsigned blocks = (unsigned)((n + kWarpsPerCta - 1) / kWarpsPerCta);
        if (P->kind == 0 && P->poly_degree > 0) {
            const unsigned pb = (unsigned)((n + kPolyWarps - 1) / kPolyWarps);
            const size_t sm = sizeof(PolyWarpSmem) * kPolyWarps;
#define E2E_POLY_CASE(DEG)                                                                                              \
    case DEG:                                                                                                           \
        render_poly_kernel<DEG><<<pb, kPolyWarps * 32, sm, stream>>>(d_x, d_y, d_w, pl->d_strips, d_item_list + i0, n, \
                                                                     P->poly, d_frame, F->view.nx, F->view.ny);        \
        break;
            switch (P->poly_degree) {
                E2E_POLY_CASE(10) E2E_POLY_CASE(12) E2E_POLY_CASE(14) E2E_POLY_CASE(16) E2E_POLY_CASE(20) E2E_POLY_CASE(24)
                default: return fail(E2E_ERR_UNSUPPORTED, "render: no kernel for this polynomial degree");
            }
#undef E2E_POLY_CASE
        } else if (P->kind == 0) {
            // the attribute is per device: set it before every launch (cheap) rather than once per process
            cudaError_t attr = cudaFuncSetAttribute(render_analytic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_an);
            if (attr != cudaSuccess) return fail_cuda(attr, "cudaFuncSetAttribute(render_analytic_kernel)");
            render_analytic_kernel<<<blocks, kWarpsPerCta * 32, smem_an, stream>>>(d_x, d_y, d_w, pl->d_strips, d_item_list + i0, n,
                                                                                   P->an, d_frame, F->view.nx, F->view.ny);
        } else if (use_tabcell) {
            const unsigned pb = (unsigned)((n + kTcWarps - 1) / kTcWarps);
            const size_t sm = 8 * tabcell_warp_smem_doubles(P->tab.os) * kTcWarps;
            cudaError_t attr = cudaFuncSetAttribute(render_tabcell_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
            if (attr != cudaSuccess) return fail_cuda(attr, "cudaFuncSetAttribute(render_tabcell_kernel)");
            render_tabcell_kernel<<<pb, kTcWarps * 32, sm, stream>>>(d_x, d_y, d_w, pl->d_strips, d_item_list + i0, n, P->tab,
                                                                     d_frame, F->view.nx, F->view.ny);
        } else
            render_tabulated_kernel<<<blocks, kWarpsPerCta * 32, smem_tab, stream>>>(d_x, d_y, d_w, pl->d_strips, d_item_list + i0,
                                                                                     n, P->tab, lat_ld, d_frame, F->view.nx, F->view.ny);
        count_launch();
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail_cuda(e, "render kernel launch");
    }
    return E2E_OK;
}

}  // namespace e2e

extern "C" {

int e2e_render_workspace_bytes(const e2e_format_t* fmt, const e2e_psf_t* psf, size_t* bytes)
{
    if (!fmt || !psf || !bytes) return fail(E2E_ERR_INVALID_ARG, "render_workspace_bytes: NULL argument");
    if (psf->nx != fmt->view.nx || psf->ny != fmt->view.ny)
        return fail(E2E_ERR_INVALID_ARG, "render_workspace_bytes: psf was created for another detector size");
    e2e_plan* pl = nullptr;
    int rc = build_plan(const_cast<e2e_format*>(fmt), psf, &pl);
    if (rc) return rc;
    *bytes = sample_arrays_bytes(fmt, psf, pl) + ctrl_bytes(pl) + cell_bytes(fmt, psf, pl);
    return E2E_OK;
}

int e2e_setup_samples(const e2e_format_t* fmt, const e2e_spectrum_t* spectrum, int32_t fiber, int32_t order_index,
                      double* d_lam, double* d_x, double* d_y, double* d_w, int64_t capacity, void* cuda_stream)
{
    if (!fmt || !spectrum) return fail(E2E_ERR_INVALID_ARG, "setup_samples: NULL argument");
    if (fiber < 0 || fiber >= fmt->view.n_fibers || order_index < 0 || order_index >= fmt->view.n_orders)
        return fail(E2E_ERR_INVALID_ARG, "setup_samples: fiber / order out of range");
    if (!spectrum->d_flux || spectrum->n < 2 || !(spectrum->dlam > 0.0) || !(spectrum->doppler > 0.0))
        return fail(E2E_ERR_INVALID_ARG, "setup_samples: bad spectrum descriptor");
    const long long N = fmt->nsamp[order_index];
    if (capacity < N) return fail(E2E_ERR_INVALID_ARG, "setup_samples: capacity smaller than the order's sample count");
    if (N == 0) return E2E_OK;
    // a one-strip launch: the strip travels as a kernel parameter, nothing is allocated and nothing synchronises
    SpectraParam sp;
    memset(&sp, 0, sizeof(sp));
    sp.s[fiber] = *spectrum;
    dim3 grid((unsigned)((N + 255) / 256), 1);
    setup_samples_kernel<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(fmt->view, sp, nullptr, fiber * fmt->view.n_orders + order_index,
                                                                      d_lam, d_x, d_y, d_w, nullptr, Strip{0, N});
    count_launch();
    cudaError_t ce = cudaGetLastError();
    if (ce != cudaSuccess) return fail_cuda(ce, "setup_samples_kernel launch");
    return E2E_OK;
}

int e2e_render_frame(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra, double* d_frame,
                     int32_t accumulate, void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!fmt || !psf || !d_frame) return fail(E2E_ERR_INVALID_ARG, "render_frame: NULL argument");
    if (psf->nx != fmt->view.nx || psf->ny != fmt->view.ny)
        return fail(E2E_ERR_INVALID_ARG, "render_frame: psf was created for another detector size");
    int rc = check_spectra(fmt, spectra, "render_frame");
    if (rc) return rc;
    e2e_plan* pl = nullptr;
    rc = build_plan(const_cast<e2e_format*>(fmt), psf, &pl);
    if (rc) return rc;
    const size_t per = sample_array_bytes(pl->total_samples);
    if (!d_workspace || ((uintptr_t)d_workspace & 255) != 0) return fail(E2E_ERR_WORKSPACE, "render_frame: workspace NULL or not 256-byte aligned");
    const size_t arrays = sample_arrays_bytes(fmt, psf, pl);
    if (workspace_bytes < arrays + ctrl_bytes(pl) + cell_bytes(fmt, psf, pl)) return fail(E2E_ERR_WORKSPACE, "render_frame: workspace too small");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    double* d_x = arrays ? (double*)d_workspace : nullptr;
    double* d_y = arrays ? (double*)((char*)d_workspace + per) : nullptr;
    double* d_w = arrays ? (double*)((char*)d_workspace + 2 * per) : nullptr;
    QueueSel qs;
    qs.ctrl = (unsigned*)((char*)d_workspace + arrays);
    qs.n = pl->n_items;
    const bool persistent = choose_moment(fmt, psf);
    // the two-kernel path zero-fills inside its first kernel (no separate pass over the frame) when the frame can be written
    // in 16-byte elements and the kernel has enough CTAs to do it at speed
    const bool fused_zero = !accumulate && use_split(fmt, psf, pl) && ((uintptr_t)d_frame & 15) == 0 &&
                            ((size_t)fmt->view.nx * fmt->view.ny) % 2 == 0 && pl->n_items >= 4 * 148;
    if (!accumulate && !fused_zero) {
        StageTimer tm(kStageZero, stream);
        E2E_CUDA(cudaMemsetAsync(d_frame, 0, (size_t)fmt->view.nx * fmt->view.ny * 8, stream));
    }
    {
        StageTimer tm(kStageSetup, stream);
        const long long before = g_launches.load();
        if (persistent) E2E_CUDA(ctrl_reset(pl, qs.ctrl, stream));
        // the two-kernel path fuses a1-a3 into its first kernel, which is timed as this stage
        if (use_split(fmt, psf, pl))
            rc = launch_cell_moments(fmt, psf, pl, spectra, qs.ctrl, nullptr, pl->n_items, stream, fused_zero ? d_frame : nullptr);
        else rc = launch_setup(fmt, pl, spectra, d_x, d_y, d_w, stream);
        if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_setup += g_launches.load() - before; }
        if (rc) return rc;
    }
    {
        StageTimer tm(kStageRender, stream);
        const long long before = g_launches.load();
        const int nparts = persistent ? 1 : pl->halves.n_bands;
        HostPipe* hp = nparts >= 2 ? host_pipe(pl) : nullptr;
        if (hp) {
            // phase-launched kernels: two row bands that share no pixel, rendered concurrently: the tail of one band's launch
            // (a few long items on otherwise idle SMs) overlaps the other band's work.  Fork to the library's stream and join.
            std::lock_guard<std::mutex> lk(hp->mu);
            const int np1 = pl->n_phases_all + 1;
            cudaStream_t sp[2] = {stream, hp->aux};
            cudaError_t ce = cudaEventRecord(hp->ev_start, stream);
            if (ce == cudaSuccess) ce = cudaStreamWaitEvent(hp->aux, hp->ev_start, 0);
            if (ce != cudaSuccess) return fail_cuda(ce, "render_frame: fork");
            for (int b = 0; b < 2 && !rc; ++b)
                rc = launch_render(fmt, psf, pl, d_x, d_y, d_w, d_frame, sp[b], qs, pl->halves.d_items,
                                   pl->halves.phase_off.data() + (size_t)b * np1, pl->n_phases_all);
            // join even when a launch failed: the caller's stream must not run ahead of work already forked
            ce = cudaEventRecord(hp->ev_aux_done, hp->aux);
            if (ce == cudaSuccess) ce = cudaStreamWaitEvent(stream, hp->ev_aux_done, 0);
            if (ce != cudaSuccess) return fail_cuda(ce, "render_frame: join");
        } else if (use_split(fmt, psf, pl)) {
            // second kernel of the two-kernel render: the contraction of every cell, under the ticket queue
            rc = launch_cell_flush(fmt, psf, pl, d_frame, qs.ctrl, nullptr, pl->n_items, 0, stream);
        } else {
            rc = launch_render(fmt, psf, pl, d_x, d_y, d_w, d_frame, stream, qs);
        }
        if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_render += g_launches.load() - before; g_prof_tot.n_calls += 1; }
    }
    return rc;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// e2e_render_frame_noalloc: the two-kernel render with its scratch (queue control block + cell records) in a file-scope device
// array instead of a caller workspace, for callers that cannot allocate.  The array exists once per GPU that loads the
// library, for the life of the process.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[E2E_NOALLOC_SCRATCH_BYTES];

// In host code `g_noalloc_scratch` is a host-side stand-in for the symbol, not a device address: the kernels get the address
// cudaGetSymbolAddress returns, resolved once per device with that device current.
static int noalloc_scratch_ptr(unsigned char** out)
{
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static unsigned char* ptr[kMaxDev] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "render_frame_noalloc: cudaGetDevice");
    if (dev < 0 || dev >= kMaxDev) return fail(E2E_ERR_UNSUPPORTED, "render_frame_noalloc: device ordinal above 63");
    std::lock_guard<std::mutex> lk(mu);
    if (!ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return fail_cuda(e, "render_frame_noalloc: cudaGetSymbolAddress");
        if (!p || ((uintptr_t)p & 255) != 0) return fail(E2E_ERR_CUDA, "render_frame_noalloc: scratch symbol has no aligned device address");
        ptr[dev] = (unsigned char*)p;
    }
    *out = ptr[dev];
    return E2E_OK;
}

// the cached schedule of (format, psf), or nullptr: a lookup only (build_plan would allocate)
static e2e_plan* find_plan(e2e_format* F, const e2e_psf* P)
{
    std::lock_guard<std::mutex> lock(F->plan_mu);
    const int nyb_key = (P->kind == 0 && P->moment_npt > 0 && !P->is_map) ? P->mom.nyb : 0;
    for (auto& p : F->plans)
        if (p->hbx == P->hbx && p->hby == P->hby && p->nyb == nyb_key) return p.get();
    return nullptr;
}

extern "C" {

int e2e_render_frame_noalloc(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra, double* d_frame,
                             int32_t accumulate, void* cuda_stream)
{
    if (!fmt || !psf || !d_frame) return fail(E2E_ERR_INVALID_ARG, "render_frame_noalloc: NULL argument");
    if (psf->nx != fmt->view.nx || psf->ny != fmt->view.ny)
        return fail(E2E_ERR_INVALID_ARG, "render_frame_noalloc: psf was created for another detector size");
    int rc = check_spectra(fmt, spectra, "render_frame_noalloc");
    if (rc) return rc;
    e2e_plan* pl = find_plan(const_cast<e2e_format*>(fmt), psf);
    if (!pl)
        return fail(E2E_ERR_UNSUPPORTED, "render_frame_noalloc: no cached schedule for this (format, psf): call e2e_render_workspace_bytes "
                                         "once at set-up (that call builds it and allocates)");
    if (!use_split(fmt, psf, pl))
        return fail(E2E_ERR_UNSUPPORTED, "render_frame_noalloc: only the two-kernel analytic render (dense sampling, constant analytic PSF) "
                                         "has a no-allocation form");
    const size_t need = ctrl_bytes(pl) + cell_bytes(fmt, psf, pl);
    if (need > (size_t)E2E_NOALLOC_SCRATCH_BYTES)
        return fail(E2E_ERR_WORKSPACE, "render_frame_noalloc: this frame needs " + std::to_string(need) + " bytes of scratch, the static array holds " +
                                           std::to_string((size_t)E2E_NOALLOC_SCRATCH_BYTES) + " (E2E_NOALLOC_SCRATCH_BYTES): use e2e_render_frame");
    unsigned char* scratch = nullptr;
    rc = noalloc_scratch_ptr(&scratch);
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    unsigned* ctrl = (unsigned*)scratch;
    // the array keeps the last call's contents: the control block is rewritten from the plan's template here, and
    // cell_moment_kernel writes every cell record cell_flush_kernel reads
    const bool fused_zero = !accumulate && ((uintptr_t)d_frame & 15) == 0 && ((size_t)fmt->view.nx * fmt->view.ny) % 2 == 0 &&
                            pl->n_items >= 4 * 148;
    if (!accumulate && !fused_zero) E2E_CUDA(cudaMemsetAsync(d_frame, 0, (size_t)fmt->view.nx * fmt->view.ny * 8, stream));
    E2E_CUDA(ctrl_reset(pl, ctrl, stream));
    rc = launch_cell_moments(fmt, psf, pl, spectra, ctrl, nullptr, pl->n_items, stream, fused_zero ? d_frame : nullptr);
    if (rc) return rc;
    return launch_cell_flush(fmt, psf, pl, d_frame, ctrl, nullptr, pl->n_items, 0, stream);
}

int e2e_render_frames_workspace_bytes(const e2e_format_t* fmt, const e2e_psf_t* psf, int32_t n_frames, size_t* bytes)
{
    if (n_frames < 1 || n_frames > 65535) return fail(E2E_ERR_INVALID_ARG, "render_frames_workspace_bytes: n_frames must be 1..65535");
    size_t one = 0;
    int rc = e2e_render_workspace_bytes(fmt, psf, &one);
    if (rc) return rc;
    e2e_plan* pl = nullptr;
    rc = build_plan(const_cast<e2e_format*>(fmt), psf, &pl);
    if (rc) return rc;
    const size_t ptr_bytes = align_up(sizeof(double*) * (size_t)n_frames, 256);
    if (use_split(fmt, psf, pl)) *bytes = batch_layout(psf, pl, n_frames, ptr_bytes).bytes;   // no per-sample arrays on this path
    else *bytes = sample_array_bytes(pl->total_samples) * (2 + (size_t)n_frames) + ptr_bytes + ctrl_bytes(pl) * (size_t)n_frames;
    return E2E_OK;
}

int e2e_render_frames(const e2e_format_t* fmt, const e2e_psf_t* psf, int32_t n_frames, const e2e_spectrum_t* spectra,
                      double* const* d_frames, int32_t accumulate, void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!fmt || !psf || !d_frames) return fail(E2E_ERR_INVALID_ARG, "render_frames: NULL argument");
    if (n_frames < 1 || n_frames > 65535) return fail(E2E_ERR_INVALID_ARG, "render_frames: n_frames must be 1..65535");
    if (psf->nx != fmt->view.nx || psf->ny != fmt->view.ny)
        return fail(E2E_ERR_INVALID_ARG, "render_frames: psf was created for another detector size");
    const int nf = fmt->view.n_fibers;
    for (int b = 0; b < n_frames; ++b) {
        if (!d_frames[b]) return fail(E2E_ERR_INVALID_ARG, "render_frames: NULL frame pointer");
        for (int c = 0; c < b; ++c)
            if (d_frames[c] == d_frames[b]) return fail(E2E_ERR_INVALID_ARG, "render_frames: two frames share one buffer");
        int rc = check_spectra(fmt, spectra ? spectra + (size_t)b * nf : nullptr, "render_frames");
        if (rc) return rc;
    }
    e2e_plan* pl = nullptr;
    int rc = build_plan(const_cast<e2e_format*>(fmt), psf, &pl);
    if (rc) return rc;
    const size_t per = sample_array_bytes(pl->total_samples);
    const size_t ptr_bytes = align_up(sizeof(double*) * (size_t)n_frames, 256);
    const bool split = use_split(fmt, psf, pl);
    const BatchLayout BL = split ? batch_layout(psf, pl, n_frames, ptr_bytes) : BatchLayout{};
    const size_t need = split ? BL.bytes : per * (2 + (size_t)n_frames) + ptr_bytes + ctrl_bytes(pl) * (size_t)n_frames;
    if (!d_workspace || ((uintptr_t)d_workspace & 255) != 0) return fail(E2E_ERR_WORKSPACE, "render_frames: workspace NULL or not 256-byte aligned");
    if (workspace_bytes < need) return fail(E2E_ERR_WORKSPACE, "render_frames: workspace too small");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    if (split) {
        // two-kernel form, the frames interleaved in one grid: the moments of every frame's cells (each frame's own spectra; a1 and a3 are recomputed
        // per frame inside the kernel, a few instructions next to a2), then ONE flush launch with one ticket queue per frame
        char* base = (char*)d_workspace;
        double** d_ptrs = (double**)base;
        SpectraParam* d_sp = (SpectraParam*)(base + BL.sp_off);
        unsigned* d_ctrl = (unsigned*)(base + BL.ctrl_off);
        CellStore cs;
        cs.cell_off = pl->d_cell_off;
        cs.hdr = (CellHeader*)(base + BL.hdr_off);
        cs.mom = (double*)(base + BL.mom_off);
        cs.frame_cells = std::max<long long>(pl->n_cells, 1);
        cs.n_frames = n_frames;
        std::vector<SpectraParam> sp((size_t)n_frames);
        memset(sp.data(), 0, sizeof(SpectraParam) * sp.size());
        for (int b = 0; b < n_frames; ++b)
            for (int f = 0; f < nf; ++f) sp[(size_t)b].s[f] = spectra[(size_t)b * nf + f];
        // pageable sources: both copies are staged before cudaMemcpyAsync returns, so neither array needs to outlive the call
        E2E_CUDA(cudaMemcpyAsync(d_ptrs, d_frames, sizeof(double*) * (size_t)n_frames, cudaMemcpyHostToDevice, stream));
        E2E_CUDA(cudaMemcpyAsync(d_sp, sp.data(), sizeof(SpectraParam) * sp.size(), cudaMemcpyHostToDevice, stream));
        for (int b = 0; b < n_frames; ++b) E2E_CUDA(ctrl_reset(pl, (unsigned*)((char*)d_ctrl + ctrl_bytes(pl) * (size_t)b), stream));
        if (!accumulate) {
            StageTimer tm(kStageZero, stream);
            for (int b = 0; b < n_frames; ++b)
                E2E_CUDA(cudaMemsetAsync(d_frames[b], 0, (size_t)fmt->view.nx * fmt->view.ny * 8, stream));
        }
        StageTimer tm(kStageRender, stream);
        const long long before = g_launches.load();
        rc = launch_cells_batch(fmt, psf, pl, n_frames, d_sp, d_ctrl, cs, d_ptrs, stream);
        if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_render += g_launches.load() - before; g_prof_tot.n_calls += 1; }
        return rc;
    }
    double* d_x = (double*)d_workspace;
    double* d_y = (double*)((char*)d_workspace + per);
    double* d_w = (double*)((char*)d_workspace + 2 * per);
    double** d_ptrs = (double**)((char*)d_workspace + per * (2 + (size_t)n_frames));
    QueueSel qs;
    qs.ctrl = (unsigned*)((char*)d_ptrs + ptr_bytes);
    qs.n = pl->n_items;
    if (choose_moment(fmt, psf))
        for (int b = 0; b < n_frames; ++b)
            E2E_CUDA(ctrl_reset(pl, (unsigned*)((char*)qs.ctrl + ctrl_bytes(pl) * (size_t)b), stream));
    // pageable source: the copy is staged before the call returns, so the caller's array need not outlive it
    E2E_CUDA(cudaMemcpyAsync(d_ptrs, d_frames, sizeof(double*) * (size_t)n_frames, cudaMemcpyHostToDevice, stream));
    if (!accumulate) {
        StageTimer tm(kStageZero, stream);
        for (int b = 0; b < n_frames; ++b)
            E2E_CUDA(cudaMemsetAsync(d_frames[b], 0, (size_t)fmt->view.nx * fmt->view.ny * 8, stream));
    }
    {
        StageTimer tm(kStageSetup, stream);
        const long long before = g_launches.load();
        for (int b = 0; b < n_frames && !rc; ++b)               // a1-a3 once (frame 0 writes x, y), a2 per frame
            rc = launch_setup(fmt, pl, spectra + (size_t)b * nf, b == 0 ? d_x : nullptr, b == 0 ? d_y : nullptr,
                              d_w + (size_t)b * (per / 8), stream);
        if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_setup += g_launches.load() - before; }
        if (rc) return rc;
    }
    {
        StageTimer tm(kStageRender, stream);
        const long long before = g_launches.load();
        rc = launch_render(fmt, psf, pl, d_x, d_y, d_w, d_frames[0], stream, qs, nullptr, nullptr, -1, n_frames, (long long)(per / 8),
                           d_ptrs, d_frames);
        if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_render += g_launches.load() - before; g_prof_tot.n_calls += 1; }
    }
    return rc;
}

int e2e_render_host_workspace_bytes(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra, size_t* bytes)
{
    if (!fmt || !psf || !spectra || !bytes) return fail(E2E_ERR_INVALID_ARG, "render_host_workspace_bytes: NULL argument");
    size_t inner = 0;
    int rc = e2e_render_workspace_bytes(fmt, psf, &inner);
    if (rc) return rc;
    const size_t npx = (size_t)fmt->view.nx * fmt->view.ny;
    size_t total = align_up(npx * 8, 256) + align_up(npx * 2, 256);       // fp64 frame + uint16 ADC frame
    for (int f = 0; f < fmt->view.n_fibers; ++f) {
        if (spectra[f].n < 2) return fail(E2E_ERR_INVALID_ARG, "render_host_workspace_bytes: bad spectrum descriptor");
        total += align_up((size_t)spectra[f].n * 8, 256);
    }
    *bytes = total + inner;
    return E2E_OK;
}

}  // extern "C"

static int check_detector_ex(const e2e_detector_ex_t* det, int32_t nx, const void* d_out, bool out16, const char* who)
{
    const std::string w(who);
    const e2e_detector_t& b = det->base;
    if (!is_fin(b.gain) || !is_fin(b.dark_e) || !is_fin(b.ron_e) || !is_fin(b.bias))
        return fail(E2E_ERR_INVALID_ARG, w + ": non-finite parameter");
    if (!is_fin(det->full_well_e) || det->full_well_e < 0.0 || !is_fin(det->e_per_adu) || det->e_per_adu < 0.0)
        return fail(E2E_ERR_INVALID_ARG, w + ": full_well_e / e_per_adu must be finite and >= 0");
    if (det->e_per_adu > 0.0 && (!is_fin(det->adu_max) || det->adu_max < 0.0))
        return fail(E2E_ERR_INVALID_ARG, w + ": adu_max must be finite and >= 0");
    if (out16 && !(det->e_per_adu > 0.0 && det->adu_max <= 65535.0))
        return fail(E2E_ERR_INVALID_ARG, w + ": the uint16 output needs e_per_adu > 0 and adu_max <= 65535");
    if ((const void*)det->d_prnu == d_out || (const void*)det->d_dark == d_out)
        return fail(E2E_ERR_INVALID_ARG, w + ": a map aliases the output frame");
    if (det->n_ports < 0) return fail(E2E_ERR_INVALID_ARG, w + ": n_ports < 0");
    if (det->xtalk && det->n_ports > 1) {
        if (det->n_ports > 16) return fail(E2E_ERR_UNSUPPORTED, w + ": more than 16 read-out ports");
        if (nx % det->n_ports != 0) return fail(E2E_ERR_UNSUPPORTED, w + ": nx is not divisible by n_ports");
        for (int i = 0; i < det->n_ports * det->n_ports; ++i)
            if (!is_fin(det->xtalk[i])) return fail(E2E_ERR_INVALID_ARG, w + ": non-finite cross-talk coupling");
    }
    return E2E_OK;
}

// HOST-buffer render: det (basic stage, fp64 electrons out), or det_ex (full stage; out16: uint16 ADC counts), or neither
static int render_frame_host_impl(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                                  const e2e_detector_t* det, const e2e_detector_ex_t* det_ex, bool out16, void* h_frame,
                                  void* d_workspace, size_t workspace_bytes, void* cuda_stream, const char* who)
{
    const std::string w(who);
    if (!fmt || !psf || !h_frame) return fail(E2E_ERR_INVALID_ARG, w + ": NULL argument");
    int rc = check_spectra(fmt, spectra, who);
    if (rc) return rc;
    size_t need = 0;
    rc = e2e_render_host_workspace_bytes(fmt, psf, spectra, &need);
    if (rc) return rc;
    if (!d_workspace || ((uintptr_t)d_workspace & 255) != 0) return fail(E2E_ERR_WORKSPACE, w + ": workspace NULL or not 256-byte aligned");
    if (workspace_bytes < need) return fail(E2E_ERR_WORKSPACE, w + ": workspace too small");
    const int nx = fmt->view.nx, ny = fmt->view.ny;
    if (det && (!is_fin(det->gain) || !is_fin(det->dark_e) || !is_fin(det->ron_e) || !is_fin(det->bias)))
        return fail(E2E_ERR_INVALID_ARG, w + ": non-finite detector parameter");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    char* p = (char*)d_workspace;
    double* d_frame = (double*)p;
    const size_t npix = (size_t)nx * ny;
    p += align_up(npix * 8, 256);
    uint16_t* d_adu = (uint16_t*)p;
    p += align_up(npix * 2, 256);
    if (det_ex) {
        rc = check_detector_ex(det_ex, nx, out16 ? (void*)d_adu : (void*)d_frame, out16, who);
        if (rc) return rc;
    }
    const size_t out_elem = out16 ? 2 : 8;
    const char* d_out = out16 ? (const char*)d_adu : (const char*)d_frame;
    const int nf = fmt->view.n_fibers;
    std::vector<e2e_spectrum_t> dev(spectra, spectra + nf);
    std::vector<int> tab_of(nf, 0);                    // fibers that share one host table share one device copy
    for (int f = 0; f < nf; ++f) {
        int same = -1;
        for (int g = 0; g < f; ++g)
            if (spectra[g].d_flux == spectra[f].d_flux && spectra[g].n == spectra[f].n) { same = g; break; }
        tab_of[f] = same >= 0 ? same : f;
        if (same >= 0) { dev[f].d_flux = dev[same].d_flux; continue; }
        dev[f].d_flux = (const double*)p;
        p += align_up((size_t)spectra[f].n * 8, 256);
    }
    // host -> device copy of the elements [lo, hi) of fiber f's table
    auto upload = [&](int f, long long lo, long long hi, cudaStream_t cs) -> cudaError_t {
        if (hi <= lo) return cudaSuccess;
        return cudaMemcpyAsync(const_cast<double*>(dev[f].d_flux) + lo, spectra[f].d_flux + lo, (size_t)(hi - lo) * 8, cudaMemcpyHostToDevice, cs);
    };
    const size_t used = (size_t)(p - (char*)d_workspace);
    e2e_plan* pl = nullptr;
    rc = build_plan(const_cast<e2e_format*>(fmt), psf, &pl);
    if (rc) return rc;
    // a6 on the rows [row0, row1) of the device frame (in place for fp64 output, into the uint16 frame otherwise)
    auto detector_rows = [&](int row0, int row1, cudaStream_t cs) -> int {
        const size_t off = (size_t)row0 * nx;
        const long long n = (long long)(row1 - row0) * nx;
        if (det_ex)
            return launch_detector_ex(d_frame + off, out16 ? (void*)(d_adu + off) : (void*)(d_frame + off), out16, n, nx, *det_ex, cs,
                                      (long long)off);
        if (det) return launch_detector(d_frame + off, d_frame + off, n, *det, cs, (long long)off);
        return E2E_OK;
    };
    HostPipe* hp = host_pipe(pl);
    const e2e_plan::BandPart& part = out16 ? pl->host16 : pl->host;   // the 2-byte output travels 4x faster: fewer, larger bands
    if (part.n_bands <= 1 || !hp) {
        // one pass: tables, render, detector, copy
        for (int f = 0; f < nf; ++f)
            if (tab_of[f] == f) E2E_CUDA(upload(f, 0, spectra[f].n, stream));
        rc = e2e_render_frame(fmt, psf, dev.data(), d_frame, 0, p, workspace_bytes - used, stream);
        if (rc) return rc;
        rc = detector_rows(0, ny, stream);
        if (rc) return rc;
        E2E_CUDA(cudaMemcpyAsync(h_frame, d_out, npix * out_elem, cudaMemcpyDeviceToHost, stream));
        E2E_CUDA(cudaStreamSynchronize(stream));
        return E2E_OK;
    }
    // banded pipeline: per row band a1-a3 of its strips, a4 + a5, a6 on the rows that became final, then those rows travel
    // to the host on the library's copy stream while the next bands render
    const size_t per = sample_array_bytes(pl->total_samples);
    const bool split = use_split(fmt, psf, pl);
    const size_t arrays = sample_arrays_bytes(fmt, psf, pl);
    if (workspace_bytes - used < arrays + ctrl_bytes(pl) + cell_bytes(fmt, psf, pl)) return fail(E2E_ERR_WORKSPACE, w + ": workspace too small");
    double* d_x = arrays ? (double*)p : nullptr;
    double* d_y = arrays ? (double*)(p + per) : nullptr;
    double* d_w = arrays ? (double*)(p + 2 * per) : nullptr;
    unsigned* d_ctrl = (unsigned*)(p + arrays);
    if (part.n_bands > kCtrlHeads) return fail(E2E_ERR_UNSUPPORTED, w + ": too many row bands");
    std::lock_guard<std::mutex> lk(hp->mu);            // one banded call at a time owns the copy stream and its events
    // bands share no pixel (build_plan): even bands on the caller's stream, odd bands on the library's second stream
    E2E_CUDA(cudaEventRecord(hp->ev_start, stream));
    E2E_CUDA(cudaStreamWaitEvent(hp->aux, hp->ev_start, 0));
    E2E_CUDA(cudaStreamWaitEvent(hp->up, hp->ev_start, 0));
    // from here on work is forked: every exit goes through the join below (errors are remembered, not returned at once)
    cudaError_t ce = cudaSuccess;
    // a2 reads of a band's samples stay inside the wavelength range of its strips (spectrum_at: elements floor(t), floor(t) + 1,
    // t = (lam / doppler - lam0) / dlam), so the tables travel on their own stream piece by piece in band order -- the part
    // band 0 reads first, then what each later band adds to the uploaded interval -- and band b waits only for its own
    // pieces.  Elements outside every band's range are read by no sample and do not travel at all.
    {
        std::vector<long long> ulo(nf, 0), uhi(nf, -1);          // uploaded interval [ulo, uhi) per table (uhi < 0: nothing yet)
        for (int b = 0; b < part.n_bands && ce == cudaSuccess; ++b) {
            for (int f = 0; f < nf && ce == cudaSuccess; ++f) {
                const double la = part.lam_lo[(size_t)b * nf + f], lb = part.lam_hi[(size_t)b * nf + f];
                if (!(la <= lb)) continue;
                const e2e_spectrum_t& sp = spectra[f];
                const int u = tab_of[f];
                const double ta = (la / sp.doppler - sp.lam0) / sp.dlam, tb = (lb / sp.doppler - sp.lam0) / sp.dlam;
                long long lo = 0, hi = sp.n;
                if (is_fin(ta) && is_fin(tb) && std::fabs(ta) < 4e18 && std::fabs(tb) < 4e18) {
                    lo = std::min<long long>(std::max<long long>((long long)std::floor(std::min(ta, tb)) - 2, 0), sp.n);
                    hi = std::max<long long>(std::min<long long>((long long)std::floor(std::max(ta, tb)) + 4, sp.n), lo);
                }
                if (hi <= lo) continue;
                if (uhi[u] < 0) { ce = upload(u, lo, hi, hp->up); ulo[u] = lo; uhi[u] = hi; continue; }
                if (lo < ulo[u]) { ce = upload(u, lo, ulo[u], hp->up); ulo[u] = lo; }
                if (hi > uhi[u] && ce == cudaSuccess) { ce = upload(u, uhi[u], hi, hp->up); uhi[u] = hi; }
            }
            if (ce == cudaSuccess) ce = cudaEventRecord(hp->ev_up[b % HostPipe::kEvents], hp->up);
        }
    }
    if (ce == cudaSuccess) ce = cudaMemsetAsync(d_frame, 0, npix * 8, stream);
    if (ce == cudaSuccess) ce = ctrl_reset(pl, d_ctrl, stream);
    // the memset and the control block must be in place before the second stream's first band
    if (ce == cudaSuccess) ce = cudaEventRecord(hp->ev_zero, stream);
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(hp->aux, hp->ev_zero, 0);
    int row0 = 0;
    for (int b = 0; b < part.n_bands && !rc && ce == cudaSuccess; ++b) {
        cudaStream_t cs = (b & 1) ? hp->aux : stream;
        ce = cudaStreamWaitEvent(cs, hp->ev_up[b % HostPipe::kEvents], 0);
        if (ce != cudaSuccess) break;
        QueueSel qs;
        qs.ctrl = d_ctrl; qs.head = b;
        qs.queue = part.d_queue + part.queue_off[b];
        qs.n = part.queue_off[b + 1] - part.queue_off[b];
        if (split) {
            // two-kernel render of this band's items: a1-a3 + moments, then the contraction under the band's queue
            rc = launch_cell_moments(fmt, psf, pl, dev.data(), d_ctrl, qs.queue, qs.n, cs);
            if (!rc) rc = launch_cell_flush(fmt, psf, pl, d_frame, d_ctrl, qs.queue, qs.n, b, cs);
        } else {
            rc = launch_setup(fmt, pl, dev.data(), d_x, d_y, d_w, cs, &part, b);   // a1-a3 of this band's strips only
            if (!rc)
                rc = launch_render(fmt, psf, pl, d_x, d_y, d_w, d_frame, cs, qs, part.d_items,
                                   part.phase_off.data() + (size_t)b * (pl->n_phases_all + 1), pl->n_phases_all);
        }
        if (rc) break;
        const int row1 = std::max(row0, part.fin_row[b]);
        if (row1 > row0) {
            rc = detector_rows(row0, row1, cs);
            if (rc) break;
            const size_t off = (size_t)row0 * nx;
            cudaEvent_t ev = hp->ev[b % HostPipe::kEvents];
            ce = cudaEventRecord(ev, cs);
            if (ce == cudaSuccess) ce = cudaStreamWaitEvent(hp->copy, ev, 0);
            if (ce == cudaSuccess)
                ce = cudaMemcpyAsync((char*)h_frame + off * out_elem, d_out + off * out_elem, (size_t)(row1 - row0) * nx * out_elem,
                                     cudaMemcpyDeviceToHost, hp->copy);
            row0 = row1;
        }
    }
    // join: the caller's stream waits for the second stream, and the call for both and for the copies
    cudaError_t cj = cudaEventRecord(hp->ev_aux_done, hp->aux);
    if (cj == cudaSuccess) cj = cudaStreamWaitEvent(stream, hp->ev_aux_done, 0);
    cudaError_t c0 = cudaStreamSynchronize(hp->up);
    cudaError_t c1 = cudaStreamSynchronize(hp->aux), c2 = cudaStreamSynchronize(stream), c3 = cudaStreamSynchronize(hp->copy);
    if (rc) return rc;
    for (cudaError_t e : {ce, cj, c0, c1, c2, c3})
        if (e != cudaSuccess) return fail_cuda(e, who);
    return E2E_OK;
}

extern "C" {

int e2e_render_frame_host(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                          const e2e_detector_t* det, double* h_frame, void* d_workspace, size_t workspace_bytes,
                          void* cuda_stream)
{
    return render_frame_host_impl(fmt, psf, spectra, det, nullptr, false, h_frame, d_workspace, workspace_bytes, cuda_stream,
                                  "render_frame_host");
}

int e2e_render_frame_host_ex(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                             const e2e_detector_ex_t* det, double* h_frame, void* d_workspace, size_t workspace_bytes,
                             void* cuda_stream)
{
    if (!det) return fail(E2E_ERR_INVALID_ARG, "render_frame_host_ex: det is NULL");
    return render_frame_host_impl(fmt, psf, spectra, nullptr, det, false, h_frame, d_workspace, workspace_bytes, cuda_stream,
                                  "render_frame_host_ex");
}

int e2e_render_frame_host_adu16(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                                const e2e_detector_ex_t* det, uint16_t* h_frame, void* d_workspace, size_t workspace_bytes,
                                void* cuda_stream)
{
    if (!det) return fail(E2E_ERR_INVALID_ARG, "render_frame_host_adu16: det is NULL");
    return render_frame_host_impl(fmt, psf, spectra, nullptr, det, true, h_frame, d_workspace, workspace_bytes, cuda_stream,
                                  "render_frame_host_adu16");
}

int e2e_apply_detector(const double* d_frame_in, double* d_frame_out, int32_t nx, int32_t ny, const e2e_detector_t* det,
                       void* cuda_stream)
{
    if (!d_frame_in || !d_frame_out || !det) return fail(E2E_ERR_INVALID_ARG, "apply_detector: NULL argument");
    if (nx <= 0 || ny <= 0) return fail(E2E_ERR_INVALID_ARG, "apply_detector: bad frame size");
    if (!is_fin(det->gain) || !is_fin(det->dark_e) || !is_fin(det->ron_e) || !is_fin(det->bias))
        return fail(E2E_ERR_INVALID_ARG, "apply_detector: non-finite parameter");
    StageTimer tm(kStageDetector, (cudaStream_t)cuda_stream);
    if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_detector += 1; }
    return launch_detector(d_frame_in, d_frame_out, (long long)nx * ny, *det, (cudaStream_t)cuda_stream);
}

int e2e_apply_detector_ex(const double* d_frame_in, double* d_frame_out, int32_t nx, int32_t ny, const e2e_detector_ex_t* det,
                          void* cuda_stream)
{
    if (!d_frame_in || !d_frame_out || !det) return fail(E2E_ERR_INVALID_ARG, "apply_detector_ex: NULL argument");
    if (nx <= 0 || ny <= 0) return fail(E2E_ERR_INVALID_ARG, "apply_detector_ex: bad frame size");
    int rc = check_detector_ex(det, nx, d_frame_out, false, "apply_detector_ex");
    if (rc) return rc;
    StageTimer tm(kStageDetector, (cudaStream_t)cuda_stream);
    if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_detector += 1; }
    return launch_detector_ex(d_frame_in, d_frame_out, false, (long long)nx * ny, nx, *det, (cudaStream_t)cuda_stream);
}

int e2e_apply_detector_adu16(const double* d_frame_in, uint16_t* d_frame_out, int32_t nx, int32_t ny, const e2e_detector_ex_t* det,
                             void* cuda_stream)
{
    if (!d_frame_in || !d_frame_out || !det) return fail(E2E_ERR_INVALID_ARG, "apply_detector_adu16: NULL argument");
    if (nx <= 0 || ny <= 0) return fail(E2E_ERR_INVALID_ARG, "apply_detector_adu16: bad frame size");
    if ((const void*)d_frame_in == (const void*)d_frame_out) return fail(E2E_ERR_INVALID_ARG, "apply_detector_adu16: in aliases out");
    int rc = check_detector_ex(det, nx, d_frame_out, true, "apply_detector_adu16");
    if (rc) return rc;
    StageTimer tm(kStageDetector, (cudaStream_t)cuda_stream);
    if (tm.on) { std::lock_guard<std::mutex> lk(g_prof_mu); g_prof_tot.n_detector += 1; }
    return launch_detector_ex(d_frame_in, d_frame_out, true, (long long)nx * ny, nx, *det, (cudaStream_t)cuda_stream);
}

// Test hook: verifies on the device, pixel by pixel, the schedule invariants the frame's bit-reproducibility rests on
// (plan_check.cuh).  Synchronous; allocates an int32 owner frame and frees it before returning.
int e2e_plan_check(const e2e_format_t* fmt, const e2e_psf_t* psf, e2e_plan_check_t* out)
{
    if (!fmt || !psf || !out) return fail(E2E_ERR_INVALID_ARG, "plan_check: NULL argument");
    if (psf->nx != fmt->view.nx || psf->ny != fmt->view.ny) return fail(E2E_ERR_INVALID_ARG, "plan_check: psf was created for another detector size");
    memset(out, 0, sizeof(*out));
    e2e_plan* pl = nullptr;
    int rc = build_plan(const_cast<e2e_format*>(fmt), psf, &pl);
    if (rc) return rc;
    const size_t npix = (size_t)fmt->view.nx * fmt->view.ny;
    int* owner = nullptr;
    PlanCheckCounters* d_cnt = nullptr;
    unsigned* d_ctrl = nullptr;
    E2E_CUDA(cudaMalloc(&owner, npix * sizeof(int)));
    cudaError_t ce = cudaMalloc(&d_cnt, sizeof(PlanCheckCounters));
    if (ce == cudaSuccess) ce = cudaMalloc(&d_ctrl, ctrl_bytes(pl));
    auto done = [&](int code) { cudaFree(owner); if (d_cnt) cudaFree(d_cnt); if (d_ctrl) cudaFree(d_ctrl); return code; };
    if (ce != cudaSuccess) return done(fail_cuda(ce, "plan_check: cudaMalloc"));
    PlanCheckCounters h;
    auto reset = [&](bool frame) {
        cudaError_t e = cudaMemset(d_cnt, 0, sizeof(PlanCheckCounters));
        if (e == cudaSuccess && frame) e = cudaMemset(owner, 0, npix * sizeof(int));
        return e;
    };
    auto fetch = [&]() {
        cudaError_t e = cudaDeviceSynchronize();
        if (e == cudaSuccess) e = cudaMemcpy(&h, d_cnt, sizeof(h), cudaMemcpyDeviceToHost);
        return e;
    };
    QueueParam nq;
    memset(&nq, 0, sizeof(nq));
    auto stamp = [&](const Item* list, int n, int mode, int band, int min_row, const QueueParam& W) {
        if (n <= 0) return;
        const int grid = mode == 2 ? std::min(n, 148 * 32) : std::min(n, 1 << 16);
        plan_check_kernel<<<grid, 32>>>(fmt->view, pl->d_strips, list, n, mode, band, min_row, W, psf->hbx, psf->hby, owner, d_cnt);
        count_launch();
    };
#define E2E_PC(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return done(fail_cuda(e__, "plan_check")); } while (0)
    out->n_items = pl->n_items; out->n_phases = pl->n_phases; out->n_dependencies = (int64_t)pl->dep_idx.size();
    out->n_host_bands = pl->host.n_bands; out->n_device_bands = pl->halves.n_bands;
    // (1) every phase launch of the plan: items of one phase share no pixel
    for (int ph = 0; ph < pl->n_phases; ++ph) {
        E2E_PC(reset(true));
        stamp(pl->d_items + pl->phase_off[ph], pl->phase_off[ph + 1] - pl->phase_off[ph], 0, 0, 0, nq);
        E2E_PC(fetch());
        out->phase_conflicts += (int64_t)h.conflicts;
        out->claimed_px = std::max<int64_t>(out->claimed_px, (int64_t)h.claimed);
    }
    // (2) the persistent launch: whole queue, then the host path's band queues
    {
        QueueParam W;
        memset(&W, 0, sizeof(W));
        W.dep_off = pl->d_dep_off; W.dep_idx = pl->d_dep_idx; W.succ_off = pl->d_succ_off; W.succ_idx = pl->d_succ_idx; W.ctrl = d_ctrl;
        E2E_PC(reset(true));
        E2E_PC(ctrl_reset(pl, d_ctrl, nullptr));
        W.queue = nullptr; W.n = pl->n_items; W.head = 0;
        stamp(pl->d_items, pl->n_items, 2, 0, 0, W);
        E2E_PC(fetch());
        out->queue_conflicts += (int64_t)h.conflicts;
        out->claimed_px = (int64_t)h.claimed;
        E2E_PC(reset(true));
        E2E_PC(ctrl_reset(pl, d_ctrl, nullptr));
        for (const e2e_plan::BandPart* part : {&pl->host, &pl->host16}) {
            E2E_PC(reset(true));
            E2E_PC(ctrl_reset(pl, d_ctrl, nullptr));
            for (int b = 0; b < part->n_bands && b < kCtrlHeads; ++b) {
                W.queue = part->d_queue + part->queue_off[b];
                W.n = part->queue_off[b + 1] - part->queue_off[b];
                W.head = b;
                stamp(pl->d_items, W.n, 2, 0, 0, W);
            }
            E2E_PC(fetch());
            out->queue_conflicts += (int64_t)h.conflicts;
            if ((int64_t)h.claimed != out->claimed_px) out->queue_conflicts += 1;  // the band queues must cover the same pixels
        }
    }
    // (3) row bands: no pixel in two bands; no row written after it was declared final
    for (int which = 0; which < 3; ++which) {
        const e2e_plan::BandPart& part = which == 0 ? pl->halves : which == 1 ? pl->host : pl->host16;
        const int np1 = pl->n_phases_all + 1;
        E2E_PC(reset(true));
        for (int b = 0; b < part.n_bands; ++b) {
            const int i0 = part.phase_off[(size_t)b * np1], i1 = part.phase_off[(size_t)b * np1 + pl->n_phases_all];
            stamp(part.d_items + i0, i1 - i0, 1, b, b > 0 ? part.fin_row[b - 1] : 0, nq);
        }
        E2E_PC(fetch());
        if (which == 0) out->device_band_conflicts = (int64_t)h.conflicts;
        else { out->host_band_conflicts += (int64_t)h.conflicts; out->host_rows_not_final += (int64_t)h.early_rows; }
        if ((int64_t)h.claimed != out->claimed_px) out->host_band_conflicts += which >= 1, out->device_band_conflicts += which == 0;
    }
#undef E2E_PC
    return done(E2E_OK);
}

int e2e_render_kernel_info(const e2e_format_t* fmt, const e2e_psf_t* psf, const char** name, double* fma_cell, double* fma_sample)
{
    if (!fmt || !psf) return fail(E2E_ERR_INVALID_ARG, "render_kernel_info: NULL argument");
    const char* nm = choose_tabcell(psf) ? "render_tabcell_kernel" : "render_tabulated_kernel";
    double pc = 0.0, ps = 0.0;
    if (choose_moment(fmt, psf)) {
        static const char* names[] = {"", "", "render_moment_kernel<2>", "render_moment_kernel<3>", "render_moment_kernel<4>"};
        static const char* map_names[] = {"", "", "render_moment_kernel<2, map>", "render_moment_kernel<3, map>", "render_moment_kernel<4, map>"};
        static const char* split_names[] = {"", "", "cell_flush_kernel<2>", "cell_flush_kernel<3>", "cell_flush_kernel<4>"};
        static const char* wide_names[] = {"", "", "cell_flush_wide_kernel<2>", "cell_flush_wide_kernel<3>", "cell_flush_wide_kernel<4>"};
        const MomentParam& M = psf->mom;
        const int npt = psf->moment_npt, jp = (M.njt + 2) / 3, ip = (M.nit + 2) / 3;
        e2e_plan* pl = nullptr;
        const bool split = build_plan(const_cast<e2e_format*>(fmt), psf, &pl) == E2E_OK && use_split(fmt, psf, pl);
        const bool wide = split && pl->small;
        nm = wide ? wide_names[npt] : split ? split_names[npt] : psf->is_map ? map_names[npt] : names[npt];
        const double nodes = psf->is_map ? (M.gx > 1 ? 2.0 : 1.0) * (M.gy > 1 ? 2.0 : 1.0) : 1.0;
        // step 2 is redone for every column panel; tiles are 8 wide, power tiles 8 deep (render_moment.cuh)
        pc = nodes * 256.0 * M.T * (2.0 * npt * M.nit * jp + 2.0 * M.nit * M.njt);         // step 2 (redone per row panel) + step 3
        if (wide) pc = 256.0 * M.T * (2.0 * npt + 2.0) * M.nit * M.njt;                      // step 2 redone per 8 x 8 tile
        // step 1 (npt DMMAs per 4 samples and node) + powers: on the two-kernel path they belong to cell_moment_kernel, not to the
        // kernel named here
        ps = split ? 0.0 : nodes * 64.0 * npt + 8.0 * npt + 8.0;
        (void)ip;
    } else if (psf->kind == 0 && psf->poly_degree > 0) {
        static thread_local char buf[40];
        snprintf(buf, sizeof buf, "render_poly_kernel<%d>", psf->poly_degree);
        nm = buf;
        const PolyParam& Q = psf->poly;
        ps = (double)Q.T * ((double)Q.ncol_pad * Q.nrow_pad + (double)(psf->poly_degree + 1) * (Q.ncol_pad + Q.nrow_pad));
    } else if (psf->kind == 0) {
        nm = "render_analytic_kernel";
    }
    if (name) *name = nm;
    if (fma_cell) *fma_cell = pc;
    if (fma_sample) *fma_sample = ps;
    return E2E_OK;
}

int e2e_render_algorithmic_fma(const e2e_format_t* fmt, const e2e_psf_t* psf, double* fma_cell, double* fma_sample)
{
    if (!fmt || !psf) return fail(E2E_ERR_INVALID_ARG, "render_algorithmic_fma: NULL argument");
    double pc = 0.0, ps = 0.0;
    if (choose_moment(fmt, psf)) {
        const double w = std::floor(2.0 * psf->hbx), h = std::floor(2.0 * psf->hby);   // nominal footprint (2 H + 1 per axis, G9)
        const double np1 = (double)psf->moment_degree + 1.0;
        const double nodes = psf->is_map ? (psf->mom.gx > 1 ? 2.0 : 1.0) * (psf->mom.gy > 1 ? 2.0 : 1.0) : 1.0;   // G21: one moment set per node
        pc = nodes * (double)psf->mom.T * (8.0 * np1 * w + 8.0 * w * h);
        ps = nodes * 8.0 * np1;
    } else if (choose_tabcell(psf)) {
        // cell-deposit method (render_tabcell.cuh): one FMA per (field node, y-offset row, x-offset, window pixel) and cell --
        // the samples of a cell sweep all os + 1 x-offsets and, on a trace flatter than 1/os px per px, 2 y-offset rows --
        // and 4 deposit products per field node and sample
        const TabParam& T = psf->tab;
        const double nodes = (T.gx > 1 ? 2.0 : 1.0) * (T.gy > 1 ? 2.0 : 1.0);
        pc = nodes * 2.0 * (double)(T.os + 1) * (double)(T.npix + 1) * (double)(T.npix + 1);
        ps = 4.0 * nodes;
    }
    if (fma_cell) *fma_cell = pc;
    if (fma_sample) *fma_sample = ps;
    return E2E_OK;
}

int e2e_measure_fp64_peak(int32_t repeats, double* burst_dfma_per_s, double* sustained_dfma_per_s)
{
    return measure_fp64_peak(repeats, burst_dfma_per_s, sustained_dfma_per_s);
}

int e2e_probe_fp64_pipe(double* results6)
{
    if (!results6) return fail(E2E_ERR_INVALID_ARG, "probe_fp64_pipe: NULL argument");
    return probe_fp64_pipe(results6);
}

int e2e_profile_enable(int32_t on)
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_on = on != 0;
    return E2E_OK;
}

int e2e_profile_read(e2e_profile_t* out, int32_t reset)
{
    if (!out) return fail(E2E_ERR_INVALID_ARG, "profile_read: out is NULL");
    std::lock_guard<std::mutex> lk(g_prof_mu);
    for (auto& p : g_prof_pending) {
        cudaError_t e = cudaEventSynchronize(p.b);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p.a, p.b);
        g_prof_free.push_back(p.a);
        g_prof_free.push_back(p.b);
        if (e != cudaSuccess) { g_prof_pending.clear(); return fail_cuda(e, "profile_read"); }
        switch (p.stage) {
            case kStageZero: g_prof_tot.ms_zero += ms; break;
            case kStageSetup: g_prof_tot.ms_setup += ms; break;
            case kStageRender: g_prof_tot.ms_render += ms; break;
            default: g_prof_tot.ms_detector += ms; break;
        }
    }
    g_prof_pending.clear();
    *out = g_prof_tot;
    if (reset) g_prof_tot = e2e_profile_t{};
    return E2E_OK;
}

}  // extern "C"
