/*
 * e2e.h -- C ABI of libe2e: B200-native echellogram rendering (sm_100a).
 *
 * The one data-parallel hot path of the end-to-end spectrograph simulator of Genoni, Landoni et al.
 * (arXiv 2008.05858; PAPER.md, cited as P:line): the Image Simulation Module,
 *
 *     "The final image of the echellogram is obtained as a superposition of individual spectral
 *      images of the fiber sampled on a proper wavelength grid.  Those are estimated as a surface
 *      integral of the convolution between the spatial profile of the fiber and the PSF ..."
 *
 *   frame[j][i] = sum_f sum_m sum_k  w_{f,m,k} * P(i - x_{f,m,k}, j - y_{f,m,k})
 *
 * over fibers f, echelle orders m and oversampled wavelength samples k.  Steps (the
 * readings of the paper they rest on are listed in DESIGN.md):
 *   a1  lam_k = lam_min + (k + 1/2) dlam,  N_m = ceil(samples_per_px * |x(lam_max) - x(lam_min)|)
 *   a2  w_k   = scale_f * S_f(lam_k / doppler_f) * E_m(lam_k) * T(lam_k) * dlam
 *   a3  (x_k, y_k) = spectral-format polynomials in (lam, m) + per-fiber offset
 *   a4  P = pixel-integrated (fiber image (x) optical PSF), analytic or tabulated
 *   a5  accumulate into the fp64 frame
 *   a6  optional detector stage: Poisson photon noise + gaussian read noise
 *
 * Conventions: pixel (i, j) = column i (x, main dispersion), row j (y, cross dispersion); it covers
 * [i-1/2, i+1/2) x [j-1/2, j+1/2); frames are row-major, frame[j*nx + i], fp64.
 *
 * Every function returns 0 (E2E_OK) or a negative error code; e2e_last_error() gives a message for
 * the last failing call of the calling thread.  Nothing aborts, throws or prints.  Pointers are HOST
 * pointers unless the name starts with d_ (DEVICE pointer, same CUDA device as the handles).
 * There is no CPU fallback: without a CUDA device every call that needs one returns E2E_ERR_CUDA.
 */
#ifndef E2E_H
#define E2E_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define E2E_API __attribute__((visibility("default")))
#else
#define E2E_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

enum {
    E2E_OK = 0,
    E2E_ERR_INVALID_ARG = -1,    /* NULL pointer, bad shape, NaN, negative sigma ... */
    E2E_ERR_NOT_MONOTONIC = -2,  /* x(lam) is not strictly monotone inside an order */
    E2E_ERR_CUDA = -3,           /* a CUDA runtime call failed (message holds cudaGetErrorString) */
    E2E_ERR_NOMEM = -4,
    E2E_ERR_UNSUPPORTED = -5,    /* valid input outside what the kernels handle (limits below) */
    E2E_ERR_WORKSPACE = -6       /* workspace pointer NULL / misaligned / too small */
};

/* message for the last failing call of this thread ("" if none); pointer valid until the next call */
E2E_API const char* e2e_last_error(void);
/* library version string, e.g. "e2e-b200 0.1 sm_100a" */
E2E_API const char* e2e_version(void);

/* ------------------------------------------------------------------------------------------------
 * Spectral format + efficiency ("spectral format data", P:165 blaze and throughput)
 * ------------------------------------------------------------------------------------------------ */
typedef struct e2e_format e2e_format_t; /* opaque; immutable after create */

typedef struct {
    int32_t nx, ny;                 /* detector size in pixels */
    int32_t n_orders;
    const int32_t* order_m;         /* [n_orders] echelle order numbers m */
    const double* lam_min;          /* [n_orders] wavelength range rendered per order, lam_min < lam_max */
    const double* lam_max;
    int32_t n_fibers;
    const double* fiber_dx;         /* [n_fibers] offsets of each fiber image in px */
    const double* fiber_dy;
    int32_t deg_l, deg_m;           /* tensor degree of the format polynomials, each 0..5 */
    const double* coef_x;           /* [(deg_l+1)*(deg_m+1)], c[p*(deg_m+1)+q] multiplies L^p M^q */
    const double* coef_y;
    double lam0, inv_dlam;          /* L = (lam - lam0) * inv_dlam */
    double m0, inv_dm;              /* M = (m - m0) * inv_dm */
    const double* blaze_lam_c;      /* [n_orders] blaze wavelength: E = amp * sinc^2(pi m (lam_c/lam - 1)) */
    const double* blaze_amp;        /* [n_orders] or NULL (= 1) */
    const double* eff_table;        /* optional common throughput T(lam) on a uniform grid, linear interp; NULL = 1 */
    int64_t eff_n;
    double eff_lam0, eff_dlam;
    double samples_per_px;          /* wavelength samples per pixel of dispersion */
} e2e_format_desc_t;

/* Copies everything (caller keeps ownership of the arrays).  Evaluates every sample position once on the
 * device to (i) check that x(lam_k) is strictly monotone in k inside each order, (ii) record the smallest
 * sample spacing and the row range of each order per 64-column bin (used to schedule renders so that concurrent warps never share a pixel).
 * Polynomial evaluation is the fixed fma-Horner sequence of DESIGN.md "O2" (inner over q=deg_m..0 in M,
 * outer over p=deg_l..0 in L), bit-identical on host and device. */
E2E_API int e2e_format_create(e2e_format_t** out, const e2e_format_desc_t* desc);
E2E_API void e2e_format_destroy(e2e_format_t* fmt);

/* number of wavelength samples: per order (same for every fiber) into n_per_order[n_orders] (may be NULL),
 * and the total over orders AND fibers into *n_total (may be NULL) */
E2E_API int e2e_format_num_samples(const e2e_format_t* fmt, int64_t* n_per_order, int64_t* n_total);

/* ------------------------------------------------------------------------------------------------
 * Parametric Spectrograph Unit ("the Parametric Version ... requires only geometrical parameters (such as dispersing
 * elements working angle, optical elements working F-Number) to recover the expected spectral format required for rendering
 * the image"; P:165 blaze "for each order"; P:59 / P:155 line tilt).  HOST code, no device call: fills the arrays an
 * e2e_format_desc_t / e2e_psf_desc_t needs from the relations of a cross-dispersed echelle spectrograph (G22):
 *   echelle   m lam = d cos(gamma) (sin alpha + sin beta), alpha = blaze + theta, blaze peak at beta_c = blaze - theta,
 *             lam_c(m) = K / m with K = 2 d cos(gamma) sin(blaze) cos(theta); one free spectral range per order,
 *             lam in [K / (m + 1/2), K / (m - 1/2)]; x = x_c + F tan(beta - beta_c), F = f_cam / pixel
 *   cross-disperser  first-order grating in Littrow at xd_lam_ref: sin beta_x = lam / d_x - sin alpha_x;
 *             y = y_c + F tan(beta_x - alpha_x)
 *   fibers    image widths Dy = core f_cam / (f_coll pixel), Dx = Dy cos(alpha) / cos(beta_c); fiber at height h along the
 *             pseudo-slit: dy = h f_cam / (f_coll pixel), dx = tan(chi) dy, tan(chi) = tan(gamma) (sin alpha + sin beta_c) / cos(beta_c)
 *   blaze     amplitude min(1, cos(alpha) / cos(beta_c)) (groove shadowing), sinc^2 profile of e2e_format_desc_t
 * x and y are delivered as the degree-(5, 5) tensor polynomials of e2e_format_desc_t (x depends on (lam, m) through
 * m lam / K - 1 only, bilinear in (L, M): its degree-5 Chebyshev interpolant is expanded exactly; y: degree-5 interpolant in
 * L); residual_x_px / residual_y_px = largest deviation of the stored polynomials from the closed forms over all orders.
 * Output arrays are owned by the caller: order arrays of capacity_orders >= m_hi - m_lo + 1 entries, coef_x / coef_y of 36,
 * fiber_dx / fiber_dy of n_fibers.  Errors: NULL / non-finite / non-positive parameters -> E2E_ERR_INVALID_ARG; a diffraction
 * angle beyond 90 degrees -> E2E_ERR_UNSUPPORTED.
 * ------------------------------------------------------------------------------------------------ */
typedef struct {
    double groove_um;               /* echelle groove spacing d (1000 / grooves per mm) */
    double blaze_deg;               /* blaze angle */
    double theta_deg;               /* in-plane angle between the incident beam and the blaze normal (quasi-Littrow: small) */
    double gamma_deg;               /* off-plane angle (gives the line tilt) */
    double xd_groove_um;            /* cross-disperser groove spacing */
    double xd_lam_ref;              /* Angstrom: cross-disperser in Littrow here; this wavelength lands on row y_c */
    double f_cam_mm, f_coll_mm;     /* camera and collimator focal lengths */
    double pixel_um;
    double fiber_core_um;           /* diameter of the fiber core as seen at the spectrograph entrance */
    int32_t m_lo, m_hi;             /* echelle orders to generate */
    double x_c, y_c;                /* column of the blaze peaks, row of xd_lam_ref */
    int32_t n_fibers;
    const double* fiber_height_um;  /* [n_fibers] positions along the pseudo-slit */
} e2e_spectrograph_t;

typedef struct {
    int32_t capacity_orders;        /* in: length of the order arrays below */
    int32_t n_orders, deg_l, deg_m; /* out */
    int32_t* order_m;               /* out [n_orders] */
    double *lam_min, *lam_max, *blaze_lam_c, *blaze_amp;   /* out [n_orders] */
    double *coef_x, *coef_y;        /* out [36] */
    double lam0, inv_dlam, m0, inv_dm;
    double *fiber_dx, *fiber_dy;    /* out [n_fibers] */
    double fiber_dx_px, fiber_dy_px;/* out: full widths of the fiber image (e2e_psf_desc_t) */
    double residual_x_px, residual_y_px;
    double x_min, x_max, y_min, y_max;   /* extent of the traces (base trace, no fiber offset) */
    double tilt_tan, K, px_per_radian;
} e2e_spectrograph_format_t;
E2E_API int e2e_spectrograph_format(const e2e_spectrograph_t* sp, e2e_spectrograph_format_t* out);

/* ------------------------------------------------------------------------------------------------
 * Instrument PSF = fiber image (x) optical PSF
 * ------------------------------------------------------------------------------------------------ */
typedef struct e2e_psf e2e_psf_t; /* opaque; immutable after create */

typedef struct {
    int32_t kind;                   /* 0 analytic: uniform ellipse (x) axis-aligned gaussian; 1 tabulated */
    double fiber_dx_px, fiber_dy_px;/* kind 0: full widths of the fiber image, main / cross dispersion; 0,0 = pure gaussian */
    double sigma_x, sigma_y;        /* kind 0: optical PSF sigmas in px ("asymmetric Gaussian"), > 0 */
    double support_nsigma;          /* kind 0: t of the footprint rule H = D/2 + t*sigma (G9); <= 0 selects 7.5 */
    int32_t n_nodes;                /* kind 0: chord-quadrature nodes Q; 0 = chosen from D/sigma so that the
                                       quadrature error is < 1e-12 of the PSF peak */
    int32_t tab_npix, tab_os;       /* kind 1: kernel size in px (e.g. 11) and cells per px (e.g. 8) */
    int32_t tab_gx, tab_gy;         /* kind 1: field grid of kernels across the detector (e.g. 5 x 5), each >= 1 */
    const double* tab;              /* kind 1: [gy][gx][npix*os][npix*os] cell values, every kernel sums to 1 */
    /* kind 0, analytic PSF MAP ("evaluate the optical PSF ... for each wavelength"; G21): when an_sigma_x and
     * an_sigma_y are not NULL they hold sigma at the nodes of an an_gx x an_gy grid over the detector (node (g, h) at
     * x = g (nx-1)/(an_gx-1), y = h (ny-1)/(an_gy-1)) and sigma_x / sigma_y above are ignored: the PSF of a sample is the
     * bilinear blend, at the sample's position, of the 4 surrounding node PSFs (weights clamped outside the grid); the
     * footprint box uses the largest node sigma per axis.  At most 64 nodes; rendered by the cell-moment kernel whatever the sampling. */
    int32_t an_gx, an_gy;
    const double* an_sigma_x;       /* HOST [an_gy][an_gx] */
    const double* an_sigma_y;
} e2e_psf_desc_t;

/* Limits (E2E_ERR_UNSUPPORTED beyond them): footprint (2H+2) <= 96 px per axis; Q <= 64; tab_npix*tab_os <= 256. */
E2E_API int e2e_psf_create(e2e_psf_t** out, const e2e_psf_desc_t* desc, int32_t nx, int32_t ny);
E2E_API void e2e_psf_destroy(e2e_psf_t* psf);

/* what the library derived from the description: the chord-quadrature order Q in use (1 for a pure gaussian,
 * 0 for a tabulated PSF) and the largest footprint in columns / rows (G9).  Any output pointer may be NULL. */
E2E_API int e2e_psf_info(const e2e_psf_t* psf, int32_t* n_nodes, int32_t* footprint_cols, int32_t* footprint_rows);

/* ------------------------------------------------------------------------------------------------
 * Rendering (a1-a5)
 * ------------------------------------------------------------------------------------------------ */
typedef struct {
    const double* d_flux;           /* DEVICE (or HOST for the *_host entry point) photon-flux table, uniform grid */
    int64_t n;                      /* table length, >= 2 */
    double lam0, dlam;              /* wavelength of flux[0], grid step > 0 */
    double scale;                   /* per-fiber illumination factor */
    double doppler;                 /* 1 + v/c: the fiber sees S(lam / doppler) */
} e2e_spectrum_t;

/* bytes of device scratch e2e_render_frame needs for this (format, psf): the control block of the render queue (4 B per
 * work item) and either, on the two-kernel analytic path (which never materialises the samples), one record per footprint
 * cell (32 B + 512 B per power tile: 1056 B per cell for the ESPRESSO-like PSF, 1.6 GB per frame) or, for the other
 * kernels, the per-sample arrays x, y, w of step a1-a3 (24 B per sample).  256-byte aligned workspace required. */
E2E_API int e2e_render_workspace_bytes(const e2e_format_t* fmt, const e2e_psf_t* psf, size_t* bytes);

/* a1-a3 only, for one (fiber, order): writes lam, x, y, w of its samples to DEVICE arrays of length
 * `capacity` >= that order's sample count (any of the four may be NULL).  Asynchronous on cuda_stream. */
E2E_API int e2e_setup_samples(const e2e_format_t* fmt, const e2e_spectrum_t* spectrum, int32_t fiber, int32_t order_index,
                      double* d_lam, double* d_x, double* d_y, double* d_w, int64_t capacity, void* cuda_stream);

/* a1-a5.  spectra: HOST array [n_fibers] whose d_flux members are DEVICE pointers.  d_frame: DEVICE
 * [ny*nx] fp64 row-major; accumulate = 0 overwrites it (it is zero-filled first), 1 adds to it.
 * Deterministic: the same inputs give the same bits (every pixel's additions happen in a fixed order).  Asynchronous on cuda_stream
 * (a cudaStream_t, NULL = default stream); launch errors are returned, later device faults surface at the
 * caller's next synchronisation.  The call allocates nothing on the device except, the first time a
 * (format, psf) pair is seen, the cached schedule (a few hundred KB). 
 * The analytic PSF under dense sampling renders with ONE kernel launch on cuda_stream.  The other kernels (sparse sampling,
 * sigma < ~0.3 px, tabulated PSF) enqueue part of their launches on a stream owned by the (format, psf) pair that forks from
 * and joins cuda_stream (two row bands that share no pixel are rendered concurrently); to the caller the call is ordered on
 * cuda_stream as a whole, and renders of different pairs never wait on each other's forked work. */
E2E_API int e2e_render_frame(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                     double* d_frame, int32_t accumulate, void* d_workspace, size_t workspace_bytes,
                     void* cuda_stream);

/* e2e_render_frame for callers that cannot allocate device memory or hold a workspace (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  Same arguments without the workspace: the scratch of the
 * two-kernel analytic render (queue control block + one record per footprint cell, see e2e_render_workspace_bytes) lives in
 * ONE static device array of E2E_NOALLOC_SCRATCH_BYTES bytes inside the library; every GPU that loads the library holds it
 * until the process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating routine; the frame has the bits
 * of e2e_render_frame's.  Conditions (else an error and nothing is launched):
 *   - the cached schedule of this (format, psf) pair exists: call e2e_render_workspace_bytes(fmt, psf, &n) once at set-up
 *     (that call builds it and allocates)                                                      -> E2E_ERR_UNSUPPORTED;
 *   - the pair renders with the two-kernel analytic path (analytic PSF with constant sigma, dense sampling)
 *                                                                                              -> E2E_ERR_UNSUPPORTED;
 *   - its scratch fits: n from e2e_render_workspace_bytes <= E2E_NOALLOC_SCRATCH_BYTES (frames up to ~20 000 footprint
 *     cells: a single order, not a full echellogram)                                           -> E2E_ERR_WORKSPACE.
 * Every call on a GPU shares the one array: calls that overlap on the GPU (different streams, different threads) RACE on it
 * and corrupt each other's frames -- serialise them on one stream or with events.  Nothing must be cleared by the caller:
 * each call rewrites the control block and every record it reads.  Asynchronous on cuda_stream. */
#define E2E_NOALLOC_SCRATCH_BYTES (32u << 20)   /* 32 MiB */
E2E_API int e2e_render_frame_noalloc(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                             double* d_frame, int32_t accumulate, void* cuda_stream);

/* Batch render on fixed geometry ("[the database] can be computed only once and used for
 * different simulation scenarios"): n_frames frames of the SAME format and PSF, each with its own spectra --
 * e.g. object / flat / Fabry-Perot exposures, or the Doppler-shifted copies of one spectrum (BJ "Precision/RV sweep").
 * spectra: HOST array [n_frames][n_fibers] (DEVICE tables); d_frames: HOST array of n_frames distinct DEVICE frame
 * pointers ([ny*nx] each).  Frame b equals e2e_render_frame(spectra + b * n_fibers, d_frames[b]) bit for bit.  The frames
 * are rendered by the same launches (two kernel launches for the whole batch on the two-kernel analytic path,
 * one ticket queue per frame), so small frames that cannot fill the GPU alone do so together; the kernels that materialise
 * the samples compute a1 and a3 (positions) once for the batch.  Workspace: e2e_render_frames_workspace_bytes.  Errors as
 * e2e_render_frame; n_frames outside 1..65535 or two equal frame pointers -> E2E_ERR_INVALID_ARG. */
E2E_API int e2e_render_frames_workspace_bytes(const e2e_format_t* fmt, const e2e_psf_t* psf, int32_t n_frames, size_t* bytes);
E2E_API int e2e_render_frames(const e2e_format_t* fmt, const e2e_psf_t* psf, int32_t n_frames, const e2e_spectrum_t* spectra,
                      double* const* d_frames, int32_t accumulate, void* d_workspace, size_t workspace_bytes,
                      void* cuda_stream);

/* Same as e2e_render_frame with HOST buffers: spectra[f].d_flux are HOST pointers and h_frame is a HOST
 * [ny*nx] array (pinned memory gives full PCIe speed).  The call copies the tables to the device, renders,
 * applies the detector stage a6 when det != NULL, copies the frame back and synchronises the stream before
 * returning.  Device scratch is taken from d_workspace, which must hold e2e_render_host_workspace_bytes() bytes.
 * The (fiber, order) strips are rendered in up to 8 row bands (5 for the uint16 output) that share no pixel
 * (a band starts only where a strip's first row lies above every row of the strips before it): even bands run on
 * cuda_stream, odd bands on a second stream owned by the library, and as soon as a band is done a6 runs on its rows
 * and they travel to the host on the library's copy stream.  The tables travel the other way on a fourth stream in
 * the order the bands read them -- the wavelength range of band 0's strips first, then what each later band adds --
 * and a band waits only for its own range; table elements no sample reads (outside every order's wavelength range
 * after the Doppler factor) are not copied.  The host tables and h_frame must stay valid and unchanged until the
 * call returns.  The frame is bit-reproducible call to call; against
 * e2e_render_frame it can differ in the last bit where strips overlap (the additions happen band by band).  Calls
 * on one (format, psf) pair are serialised. */
E2E_API int e2e_render_host_workspace_bytes(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                                    size_t* bytes);
struct e2e_detector;
E2E_API int e2e_render_frame_host(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                          const struct e2e_detector* det /* may be NULL */, double* h_frame, void* d_workspace,
                          size_t workspace_bytes, void* cuda_stream);

/* The same with the full detector stage (e2e_detector_ex_t below; det must not be NULL), fp64 electrons or ADC counts out. */
struct e2e_detector_ex;
E2E_API int e2e_render_frame_host_ex(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                             const struct e2e_detector_ex* det, double* h_frame, void* d_workspace, size_t workspace_bytes,
                             void* cuda_stream);
/* The same with the ADC counts delivered as uint16 (the raw frame an instrument writes, ~40 000 ADU px^-1):
 * h_frame: HOST uint16 [ny*nx]; needs det->e_per_adu > 0 and det->adu_max <= 65535.  The device-to-host copy, which bounds
 * the fp64 host path, shrinks 4x.  Element for element the value of e2e_render_frame_host_ex, cast. */
E2E_API int e2e_render_frame_host_adu16(const e2e_format_t* fmt, const e2e_psf_t* psf, const e2e_spectrum_t* spectra,
                                const struct e2e_detector_ex* det, uint16_t* h_frame, void* d_workspace,
                                size_t workspace_bytes, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Detector stage (a6; "photon noise and all other specific detector noises ... are added on the
 * final synthetic echellogram").  out[p] = (n + bias) + ron_e * z1 with mu = max(0, gain*in[p] + dark_e),
 * n ~ Poisson(mu), z1 ~ N(0,1), drawn from a Philox4x32-10 stream keyed by (seed, pixel index p = j*nx + i): the
 * result does not depend on launch geometry and is reproducible bit for bit.  Algorithm (G12, rounds 2 + 3):
 * the pixels 2q and 2q + 1 share the stream of pair q = p >> 1, and every block serves both with independent variates:
 * block 0 gives one Box-Muller pair, its cos half is z1 of the even pixel and its sin half z1 of the odd one; mu < 64:
 * n by inversion (sequential search) with the pixel's own uniform of block 1 (words 0-1 even, 2-3 odd) -- an exact Poisson
 * draw up to the 53-bit uniform, capped at n = 255 (probability < 1e-70); mu >= 64: with z2 from block 2 (formed like z1),
 * n = max(0, floor(mu + sqrt(mu) z2 + (z2^2 - 1)/6 + 1/2)), the normal approximation with the first
 * Cornish-Fisher term -- NOT an exact Poisson draw: mean mu, skewness 1/sqrt(mu) as Poisson, variance mu + 5/36
 * (0.2 % high at mu = 64, 3e-6 at 4e4 e-), and the law changes at mu = 64.
 * ------------------------------------------------------------------------------------------------ */
typedef struct e2e_detector {
    double gain, dark_e, ron_e, bias;
    uint64_t seed;
} e2e_detector_t;

/* d_frame_in / d_frame_out: DEVICE [ny*nx]; may be the same pointer.  Asynchronous on cuda_stream. */
E2E_API int e2e_apply_detector(const double* d_frame_in, double* d_frame_out, int32_t nx, int32_t ny,
                       const e2e_detector_t* det, void* cuda_stream);

/* Full detector stage ("... all other specific detector noises (e.g. dark current, RON, pixels
 * non-uniform response and cross-talk)"; readings G19 and G20 of DESIGN.md).  Per pixel p:
 *   mu = max(0, gain * prnu[p] * in[p] + dark[p]);  (z1, n) = the draws of the basic stage;
 *   e  = min(n, full_well_e) when full_well_e > 0 (the well saturates before read-out);
 *   v  = e + ron_e * z1                                                               (video signal)
 *   no cross-talk:
 *     e_per_adu <= 0:  out[p] = (e + bias) + ron_e * z1                               (electrons)
 *     e_per_adu  > 0:  out[p] = clamp(floor((v / e_per_adu + bias) + 1/2), 0, adu_max)   (ADC counts)
 *   cross-talk (xtalk != NULL and n_ports > 1; G20): the detector is read through n_ports ports, port a = columns
 *   [a W, (a+1) W), W = nx / n_ports, all clocked together; a fraction X[a][b] of the video signal of port b appears in
 *   port a at the same in-port column c:  s = v_a; for b = 0 .. n_ports-1, b != a: s = s + X[a][b] * v_b;
 *     e_per_adu <= 0:  out = s + bias;      e_per_adu > 0:  out = clamp(floor((s / e_per_adu + bias) + 1/2), 0, adu_max)
 * d_prnu (pixel response non-uniformity) and d_dark (dark electrons per pixel) are DEVICE [ny*nx] maps owned by the
 * caller, or NULL (= 1 and base.dark_e).  xtalk is a HOST [n_ports][n_ports] matrix (copied by the call; the diagonal is
 * ignored), n_ports <= 16, nx divisible by n_ports.  With both maps NULL, full_well_e = 0, e_per_adu = 0 and no
 * cross-talk the result equals e2e_apply_detector bit for bit.  Errors: NULL frame / det, non-finite or negative
 * full_well_e, e_per_adu, adu_max, a non-finite coupling -> E2E_ERR_INVALID_ARG; n_ports > 16 or nx % n_ports != 0 ->
 * E2E_ERR_UNSUPPORTED.  Asynchronous on cuda_stream; in may equal out; the maps must not alias out. */
typedef struct e2e_detector_ex {
    e2e_detector_t base;
    const double* d_prnu;
    const double* d_dark;
    double full_well_e;
    double e_per_adu;
    double adu_max;
    int32_t n_ports;                /* read-out ports for the cross-talk; 0 or 1 = none */
    const double* xtalk;            /* HOST [n_ports][n_ports] coupling X[a][b], or NULL */
} e2e_detector_ex_t;
E2E_API int e2e_apply_detector_ex(const double* d_frame_in, double* d_frame_out, int32_t nx, int32_t ny,
                          const e2e_detector_ex_t* det, void* cuda_stream);

/* The same stage with the ADC counts stored as uint16 (raw frames of ~40 000 ADU px^-1): needs
 * e_per_adu > 0 and adu_max <= 65535 (else E2E_ERR_INVALID_ARG); d_frame_out: DEVICE uint16 [ny*nx], a quarter of the
 * fp64 frame's bytes on the way to the host.  Element for element the value of e2e_apply_detector_ex, cast. */
E2E_API int e2e_apply_detector_adu16(const double* d_frame_in, uint16_t* d_frame_out, int32_t nx, int32_t ny,
                             const e2e_detector_ex_t* det, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Measurement helpers (used by bench.py; not part of the rendering path)
 * ------------------------------------------------------------------------------------------------ */
/* FP64 roofline denominator.  Launches all-SM kernels of independent fp64 chains `repeats` times back to back
 * (each launch ~10 ms), once as DFMA chains and once as mma.sync.m8n8k4.f64 (DMMA) chains -- both feed the same FP64
 * pipe -- and returns the larger rate in fused multiply-adds per second (flop/s = 2x): *burst = the fastest single
 * launch, *sustained = total work / total time of the second half of the launches.  Synchronous. */
E2E_API int e2e_measure_fp64_peak(int32_t repeats, double* burst_dfma_per_s, double* sustained_dfma_per_s);

/* Probes of one SM's FP64 pipe under the render kernel's instruction mix; results6[0] cycles per
 * mma.sync.m8n8k4.f64 (DMMA) in one dependent accumulator chain, [1] cycles per DMMA with two independent chains in one warp
 * (= the issue interval: one warp can keep its scheduler's pipe busy), [2] DMMAs per clock and SM with 16 DMMA warps (0.25 =
 * 64 fused multiply-adds per clock), [3] scalar DFMA warp instructions per clock and SM from 4 warps of independent chains
 * alone, [4] from the same 4 warps while 16 DMMA warps run next to them (scalar fp64 starves behind a saturated pipe),
 * [5] what the DMMA warps got in that mix.  Synchronous, a few milliseconds. */
E2E_API int e2e_probe_fp64_pipe(double* results6);

/* Which a4+a5 kernel e2e_render_frame launches for this (format, psf) pair and what it executes: *name is a static
 * string ("cell_flush_kernel<2>" -- the dominant kernel of the two-kernel analytic path, whose first kernel is
 * cell_moment_kernel --, "render_moment_kernel<2, map>", "render_poly_kernel<14>", "render_analytic_kernel",
 * "render_tabcell_kernel", "render_tabulated_kernel"; the batch call and the PSF map run "render_moment_kernel<NPT>");
 * *executed_fma_per_cell / *executed_fma_per_sample are the fp64 fused multiply-adds THAT kernel issues per footprint
 * cell and per sample (DMMA counted as 256), 0 where it does not apply.  Any output pointer may be NULL. */
E2E_API int e2e_render_kernel_info(const e2e_format_t* fmt, const e2e_psf_t* psf, const char** name,
                                   double* executed_fma_per_cell, double* executed_fma_per_sample);

/* Algorithmic work of the a4+a5 method e2e_render_frame uses for this pair (DESIGN.md 5.3 "Roofline"), without the
 * padding of the DMMA tiles: fp64 fused multiply-adds per footprint cell, T (8 (P+1) w + 8 w h) with w x h the nominal
 * footprint (2 H + 1 pixels per axis, G9), P the x-phase degree, T the chord terms, and per sample, 8 (P+1) (moment update;
 * on the two-kernel path the per-cell part is cell_flush_kernel's work and the per-sample part cell_moment_kernel's).
 * Tabulated PSF (cell-deposit kernel): per cell nodes x 2 y-offset rows x (os+1) x-offsets x (npix+1)^2 window
 * pixels, per sample 4 x nodes deposit products (nodes = field nodes blended per sample: 1, 2 or 4).
 * 0 for the kernels that do not work cell by cell.  Output pointers may be NULL. */
E2E_API int e2e_render_algorithmic_fma(const e2e_format_t* fmt, const e2e_psf_t* psf, double* fma_per_cell,
                                       double* fma_per_sample);

/* Test hook: verifies on the device, pixel by pixel, the invariants of the render schedule that make the frame
 * bit-reproducible although it is accumulated with L2 reductions: every footprint box (G9) of every work
 * item is stamped into an int32 owner frame and
 *   phase_conflicts        pixels claimed by two items of one phase launch (render_poly / _analytic / _tabcell / _tabulated);
 *   queue_conflicts        persistent launch (render_moment): pixels whose previous writer is not a direct dependency of the
 *                          item that writes next, run under the render kernel's own queue discipline (whole queue + the
 *                          host path's band queues); zero in one run proves every pixel's writers form a chain;
 *   device_band_conflicts  pixels shared between the two row bands the phase-launched kernels render concurrently;
 *   host_band_conflicts    pixels shared between the host path's row bands;
 *   host_rows_not_final    pixels a host band writes above the rows already declared final (copied to the host)
 * must all be 0.  claimed_px = pixels inside at least one footprint box (> 0).  Synchronous on the device; allocates and
 * frees 4 bytes per pixel. */
typedef struct {
    int64_t n_items, n_phases, n_dependencies;
    int64_t claimed_px;
    int64_t phase_conflicts, queue_conflicts, device_band_conflicts, host_band_conflicts, host_rows_not_final;
    int32_t n_host_bands, n_device_bands;
} e2e_plan_check_t;
E2E_API int e2e_plan_check(const e2e_format_t* fmt, const e2e_psf_t* psf, e2e_plan_check_t* out);

/* Number of kernel launches the library has issued since load (all entry points), for bench.py's gpu_launches. */
E2E_API int64_t e2e_launch_count(void);

/* Per-stage device timing.  While enabled, every e2e_render_frame / e2e_apply_detector call brackets its stages
 * with CUDA events recorded on the caller's stream (no synchronisation is added).  e2e_profile_read waits for
 * the recorded events, adds their elapsed times to the totals below and returns them; reset != 0 clears the
 * totals afterwards.  ms_* are summed device milliseconds, n_* the number of kernel launches in that stage. */
typedef struct {
    double ms_zero;      /* zero-fill of the frame (cudaMemsetAsync); 0 where the two-kernel path zero-fills inside cell_moment_kernel (counted in ms_setup) */
    double ms_setup;     /* a1-a3 sample-setup kernel; on the two-kernel analytic path: cell_moment_kernel (a1-a3 fused with the
                            weighted phase moments of every footprint cell) */
    double ms_render;    /* a4-a5 render kernels (all phases); on the two-kernel path: cell_flush_kernel (the contraction + a5) */
    double ms_detector;  /* a6 */
    int64_t n_setup, n_render, n_detector;
    int64_t n_calls;     /* e2e_render_frame calls covered */
} e2e_profile_t;
E2E_API int e2e_profile_enable(int32_t on);
E2E_API int e2e_profile_read(e2e_profile_t* out, int32_t reset);

#ifdef __cplusplus
}
#endif
#endif /* E2E_H */
