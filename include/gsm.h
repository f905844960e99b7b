/* gsm.h - C ABI of the B200-native Generalized Source Method (GSM) hot path.
 *
 * Method: A.A. Shcherbakov, A.V. Tishchenko, "3D periodic dielectric composite homogenization based on the
 * Generalized Source Method" (arxiv 1501.01752).  Citations "PAPER.md:<line>" refer to the text of that paper.
 *
 * What the library computes (Eq. 4, truncated to N1 x N2 x N3 harmonics):
 *
 *     E_{a,m} - sum_b G_{m;ab} sum_{m'} c_{m-m'} E_{b,m'} = a_a delta_{m,0}
 *     G_{m;ab} = (k_b^2 delta_ab - k_{a,m} k_{b,m}) / (k_m.k_m - k_b^2),   k_m = k_bloch + (m1 K1, m2 K2, m3 K3),
 *     K_a = 2 pi / Lambda_a,   k_b^2 = k0^2 eps_b,   c_d = (Delta eps / eps_b)_d  (Fourier coefficients of
 *     (eps(r) - eps_b)/eps_b, plain Laurent rule).
 *
 * The operator y = x - G (T x) is applied with a zero-padded 3-D FFT convolution and the system is
 * solved by full GMRES with modified Gram-Schmidt.  A scan over many (k_bloch, k0) points returns
 * the 0-th order response used by the pole search of Eq. 6-10.
 *
 * Conventions
 *   - All floating point is IEEE double; complex numbers are interleaved (re, im) doubles.
 *   - Units: eps0 = mu0 = c = 1, relative permittivities; "omega" is passed as the vacuum wavenumber k0 = omega/c.
 *   - Harmonic orders along axis a: m_a = i_a + mmin_a, i_a = 0..N_a-1, mmin_a = -(N_a-1)/2 for odd N_a and
 *     -N_a/2 for even N_a.  Field layout: x[batch][3][N1][N2][N3], last index fastest.
 *   - Coefficient layout (gsm_plan_coeffs): c[(2N1-1)][(2N2-1)][(2N3-1)], index d_a + N_a - 1.
 *   - Pointer arguments are HOST pointers unless the name starts with d_ (DEVICE pointer, 16-byte aligned, on the
 *     plan's device).  The caller owns every argument buffer; the plan owns all device scratch.
 *   - Work is enqueued on the plan's CUDA stream (solves of 8 or more points also use streams of the plan's own, forked
 *     from and joined to that stream with events).  gsm_apply returns without synchronising; every other call returns
 *     after the host results it writes are valid.
 *   - Errors are return codes (no exceptions, no abort, no CPU fallback).  Negative = failure, nothing valid
 *     written; positive = warning, outputs written.  gsm_last_error gives a text for the last failure.
 */
#ifndef GSM_H_
#define GSM_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gsm_plan gsm_plan; /* opaque: coefficient spectrum, FFT workspaces, Krylov pool on one device */

typedef enum {
    GSM_OK = 0,
    GSM_NOT_CONVERGED = 1,     /* max_iters reached for at least one point; best iterate and history returned */
    GSM_E_INVALID = -1,        /* bad argument (null pointer, size out of range, batch > max_batch, ...)       */
    GSM_E_ALLOC = -2,          /* host or device allocation failed                                            */
    GSM_E_CUDA = -3,           /* a CUDA runtime call or kernel launch failed                                 */
    GSM_E_SINGULAR_BASIS = -4  /* min_m |k_m.k_m - k_b^2| / |k_b^2| < 1e-12: eps_b violates PAPER.md:52       */
} gsm_status;

enum { GSM_SPHERE = 0, GSM_ELLIPSOID = 1, GSM_BOX = 2, GSM_POLYHEDRON = 3 };

/* Formulation solved by the plan.
 *   GSM_FORM_E: Eq. 4, unknown E, coefficients c_d = ((eps - eps_b)/eps_b)_d            (the default)
 *   GSM_FORM_H: Eq. 5, unknown H:
 *       H_m - k_m x [ sum_m' D_{m-m'} (k_m' x H_m') ] / (k_b^2 - k_m.k_m) = h delta_{m,0},
 *       D_d = delta_{d,0} - (eps_b/eps)_d, found analytically like c_d: background 1 - eps_b/eps_bg,
 *       each inclusion adds (eps_b/eps_bg - eps_b/eps_i) x its Fourier image (exact for non-overlapping inclusions);
 *       voxel path: transform of 1 - eps_b/eps_j.  gsm_plan_coeffs returns D_d.  `pol` is the amplitude h of H^inc. */
enum { GSM_FORM_E = 0, GSM_FORM_H = 1 };

/* Flags of a plan (gsm_plan_desc.flags, 0 in normal use).  They select an alternative code path where a default one
 * exists, so that tests can hold both to the same parity bar:
 *   GSM_FLAG_TWO_SWEEP     Gram-Schmidt by the two-sweep kernels even where one field vector fits a thread-block cluster
 *   GSM_FLAG_GENERIC_APPLY generic radix-2/4/8 FFT passes even where a 64- or 128-point fast path applies
 *   GSM_FLAG_FUSED_APPLY   64-point fast path as ONE persistent launch that keeps the z-transformed intermediate in L2
 *                          (apply_fused64.cu) instead of three launches through HBM; measured slower
 *   GSM_FLAG_SLOT_REFILL   gsm_scan from a zero start with more points than max_batch: instead of solving max_batch points,
 *                          draining, and taking the next max_batch, a slot whose solve has finished is handed the next pending
 *                          point at once (every solve at its own Arnoldi index).  Same results bit for bit; measured neutral
 *                          to slightly slower on the 31^3 workload, where the draining ticks are cheap */
enum { GSM_FLAG_TWO_SWEEP = 1, GSM_FLAG_GENERIC_APPLY = 2, GSM_FLAG_FUSED_APPLY = 4, GSM_FLAG_SLOT_REFILL = 8 };

#define GSM_MAX_ITERS 512   /* largest accepted gsm_plan_desc.max_iters */

/* One analytic inclusion ("Fourier images of sphere and polyhedron can be combined").
 * size = (R, -, -) for a sphere, semi-axes for an ellipsoid, full edge lengths for an axis-aligned box; same
 * length unit as the periods.  The inclusion's permittivity replaces the background inside it; overlapping
 * inclusions superpose their (eps_i - eps_bg) contrasts.
 * GSM_POLYHEDRON: any closed polyhedron with planar faces, convex or not (size unused).  vertices[n_vertices][3] are
 * given relative to center; face f lists face_sizes[f] >= 3 vertex indices, consecutively in face_vertices, counter-
 * clockwise seen from outside.  Its Fourier image is evaluated in closed form (divergence theorem: faces, then edges).
 * The arrays are host memory, read before gsm_plan_create / gsm_plan_set_cell return. */
typedef struct {
    int kind;
    double center[3];
    double size[3];
    double eps_re, eps_im;
    int n_vertices;
    const double* vertices;
    int n_faces;
    const int* face_sizes;
    const int* face_vertices;
} gsm_shape;

/* Plan descriptor.  Exactly one of (n_shapes > 0, shapes) or (eps_grid_host != NULL) describes the cell.
 * Voxel path: eps_grid_host[voxels[0]][voxels[1]][voxels[2]] complex, sample j at r_a = j_a Lambda_a / voxels[a];
 * 2*orders[a]-1 <= voxels[a] <= 2048.  The harmonics are the discrete Fourier transform of the grid: a
 * device FFT when every voxels[a] is a power of two <= 512, the defining sums (axis by axis) for any other size.  The
 * defining sums cost about V1 V2 V3 (2 N3 - 1) complex multiply-adds for the first axis and less for the others (5e11 for
 * 2048^3 voxels at 31 orders, where an FFT would need 1e12 / 32), read with long strides: fine for a plan built once,
 * slow for a cell that changes every step - resample such a grid to a power of two <= 512 where that matters. */
typedef struct {
    double period[3];            /* Lambda_1..3                 */
    int orders[3];               /* N1..N3 harmonics kept per axis, 1 <= N <= 256 (Table 1)       */
    double eps_bg_re, eps_bg_im; /* background permittivity of the analytic path                               */
    double eps_b_re, eps_b_im;   /* basis permittivity eps_b; must make every k_m^2 != k_b^2  */
    int n_shapes;
    const gsm_shape* shapes;
    int voxels[3];
    const double* eps_grid_host;
    int max_iters;               /* GMRES basis size (unrestarted); default 64 if <= 0; at most GSM_MAX_ITERS  */
    int max_batch;               /* (k, omega) points solved concurrently; default 1 if <= 0                   */
    void* cuda_stream;           /* cudaStream_t to enqueue on; NULL = the legacy default stream               */
    int formulation;             /* GSM_FORM_E (0) or GSM_FORM_H (1)                                           */
    int flags;                   /* GSM_FLAG_* diagnostics, 0 in normal use                                    */
} gsm_plan_desc;

/* Build the plan on the current CUDA device: evaluate c_d (analytic closed forms or FFT of the voxel grid),
 * embed it in the P1 x P2 x P3 circulant grid (P_a = smallest power of two >= 2 N_a - 1, 1 if N_a == 1), transform
 * it once, allocate workspaces for max_batch concurrent solves.  *out is NULL on failure. */
gsm_status gsm_plan_create(const gsm_plan_desc* desc, gsm_plan** out);
gsm_status gsm_plan_destroy(gsm_plan* plan);

/* Test hook: copy the coefficients c_d the plan was built from (device result) to host_out,
 * (2N1-1)(2N2-1)(2N3-1) complex numbers in the layout stated above. */
gsm_status gsm_plan_coeffs(const gsm_plan* plan, double* host_out);

/* FFT grid sizes P1..P3 chosen by the plan, device bytes held now (every workspace, including those grown on demand by
 * gsm_scan_mesh and the slot-refill scan; a voxel grid of a new size replaces the old block), and the number of kernel
 * launches enqueued so far. */
gsm_status gsm_plan_info(const gsm_plan* plan, int fft_grid[3], long long* device_bytes, long long* launches);

/* Replace the cell of an existing plan - periods, permittivities and shapes or voxel grid, i.e. step a0 (PAPER.md:62,
 * :99: the harmonics depend only on the geometry) - keeping orders, max_iters, max_batch and every workspace.
 * desc->orders must equal the plan's; voxel grids follow the rules of gsm_plan_create.  Host arrays in desc are read
 * before return and not retained. */
gsm_status gsm_plan_set_cell(gsm_plan* plan, const gsm_plan_desc* desc);

/* Launch accounting.  Every kernel the library enqueues is counted per kernel class (gsm_kernel_class_count()
 * classes, names from gsm_kernel_class_name(cls)).  gsm_plan_profile(plan, 1) additionally brackets every launch
 * with a CUDA event pair on the plan's stream; gsm_plan_profile_read synchronises the stream and returns, for the
 * first ncls classes, the launch counts, the summed device time in milliseconds and the summed algorithmic bytes
 * (the minimal reads + writes of each launch as designed) since the last reset (any array may
 * be NULL); reset != 0 clears them.  Times are zero for launches made while profiling was off. */
gsm_status gsm_plan_profile(gsm_plan* plan, int enable);
gsm_status gsm_plan_profile_read(gsm_plan* plan, int ncls, long long* launches, double* ms, double* bytes, int reset);
int gsm_kernel_class_count(void);
const char* gsm_kernel_class_name(int cls);

/* Operator apply, Eq. 4 left-hand side: y[b] = x[b] - G(k_bloch[b], k0[b]) (T x[b]), b < batch.
 * k_bloch[batch][3], k0[batch] are host arrays (copied before return).  d_x, d_y: device, [batch][3][N1][N2][N3]
 * complex; they must not overlap.  1 <= batch <= max_batch.  Asynchronous on the plan's stream. */
gsm_status gsm_apply(gsm_plan* plan, int batch, const double* k_bloch, const double* k0, const void* d_x, void* d_y);

/* One solve of Eq. 4 with right-hand side a delta_{m,0} by full GMRES from x0 = 0, stopping when
 * the residual estimate |g_{j+1}| / ||b|| <= tol.  pol = complex amplitude a (3 complex).
 * d_E_out: device, [3][N1][N2][N3] complex.  resid_hist_host (may be NULL): first min(n_iters, hist_cap) residual
 * estimates.  n_iters: iterations used.  true_rel_resid: ||b - A E|| / ||b|| recomputed with one more apply. */
gsm_status gsm_solve(gsm_plan* plan, const double k_bloch[3], double k0, const double pol[6], double tol,
                     void* d_E_out, double* resid_hist_host, int hist_cap, int* n_iters, double* true_rel_resid);

/* Residual history of one solve of the most recent lock-step batch (gsm_solve: b = 0; gsm_scan / gsm_scan_guess with
 * npts <= max_batch: b = list index; longer lists and gsm_scan_mesh run several batches, of which the last is kept):
 * the first min(n_iters, hist_cap) residual estimates |g_{j+1}| / ||b|| and *n_iters.
 * GSM_E_INVALID if b is not a solve of that batch. */
gsm_status gsm_plan_history(gsm_plan* plan, int b, double* resid_hist_host, int hist_cap, int* n_iters);

/* Scan: npts independent solves sharing the plan, run max_batch at a time in lock step.
 * resp_host[npts][3] complex = E at m = 0; iters[npts]; resid[npts] = true relative residuals.
 * d_E_out (may be NULL): device, [npts][3][N1][N2][N3] complex, all fields. */
gsm_status gsm_scan(gsm_plan* plan, int npts, const double* k_bloch, const double* k0, const double* pol,
                    double tol, double* resp_host, int* iters, double* resid, void* d_E_out);

/* gsm_scan with an initial guess per point (Saad's GMRES with x0 != 0: r0 = b - A x0, solve A d = r0, E = x0 + d; the
 * stop test stays relative to ||b||).  d_x0: device, [npts][3][N1][N2][N3] complex, or NULL (= gsm_scan); it may be the
 * same buffer as d_E_out.  A guess whose residual is not below ||b|| is ignored for that point (zero start).  The
 * reported iteration count excludes the one extra operator apply that forms r0. */
gsm_status gsm_scan_guess(gsm_plan* plan, int npts, const double* k_bloch, const double* k0, const double* pol,
                          double tol, const void* d_x0, double* resp_host, int* iters, double* resid, void* d_E_out);

/* Scan of an ORDERED mesh: the list is a line in (k, omega) space sampled at equidistant parameter values in list order
 * ("equidistant mesh kappa_p").  The points are solved in `levels` waves, coarse to fine: wave 0 takes
 * every 2^(levels-1)-th point from a zero start, each later wave the points mid-way between those already solved,
 * started from the Lagrange interpolation (the 8 nearest solved points) of their solutions (gsm_scan_guess); once a
 * guessed wave has needed at most one iteration per point on average, all remaining points form the next wave.  Where the
 * responses solved so far show poles inside the mesh (the pole search of Eq. 7-10 in units of the list index), the
 * interpolation is done on the field times prod (t - eta_k), which is smooth across a pole.  Same results as gsm_scan
 * up to the solver tolerance, fewer iterations.  levels = 1 is gsm_scan.  Outputs as gsm_scan, in list order. */
gsm_status gsm_scan_mesh(gsm_plan* plan, int npts, const double* k_bloch, const double* k0, const double* pol,
                         double tol, int levels, double* resp_host, int* iters, double* resid, void* d_E_out);

/* Host-only helper (no device work): the solve order and the interpolation stencils gsm_scan_mesh uses for a list of
 * npts points and `levels` waves.  collapse_after = c > 0: all points still unsolved after wave c form wave c + 1 (what
 * gsm_scan_mesh does once wave c needed at most one iteration per point); c <= 0: never.  wave[npts] = wave in which each
 * point is solved (0 = zero start); nodes[npts][8] = list indices of the points its guess interpolates (-1 = unused; all
 * -1 in wave 0), weights[npts][8] = their Lagrange weights in the list index (before the pole factor of gsm_scan_mesh). */
gsm_status gsm_mesh_schedule(int npts, int levels, int collapse_after, int* wave, int* nodes, double* weights);

/* Pole search, host side (Eq. 7-10, with xi in the numerator of Eq. 9 - DESIGN.md reading R11).
 * kappa[npts] equidistant and increasing, xi[npts] complex, npts >= Np + Nd.  All npts - Nd sliding windows of
 * Nd + 1 points are used (least squares).  eta[Np], zeta[Np] complex.  *best = index of the root with
 * kappa_lo <= Re eta <= kappa_hi and the largest |zeta|, or -1. */
gsm_status gsm_pole_search(int npts, const double* kappa, const double* xi, int Np, int Nd,
                           double kappa_lo, double kappa_hi, double* eta, double* zeta, int* best);

/* Retrieval of one effective index (n_eff = eta / k0, eps_eff = n_eff^2) by the two-stage scan of
 * DESIGN.md reading R16, all host orchestration around gsm_scan and gsm_pole_search:
 *   1. coarse scan: ncoarse equidistant kappa = n k0 on [n_lo, n_hi] along the unit direction dir[3] with amplitude pol
 *      (3 complex), response = component `comp` of the 0-th order field; pole search (Np = 5, Nd = 10) -> estimate eta_c;
 *   2. fine scan: nfine points with spacing fine_step * k0 centred so that eta_c falls mid-way between the two middle
 *      nodes (a sample too close to the pole spoils the fit); pole search -> eta.
 * comp = -1: response = projection of the 0-th order field on the amplitude (see gsm_retrieve_neff_many).
 * ncoarse, nfine >= 15 (= Np + Nd); nfine even.  out[0..1] = n_eff (re, im), out[2..3] = eps_eff = n_eff^2,
 * out[4..5] = pole amplitude zeta.  GSM_NOT_CONVERGED (warning) if a solve hit max_iters; GSM_E_INVALID if no pole with
 * Re eta inside the scanned window was found in either stage. */
gsm_status gsm_retrieve_neff(gsm_plan* plan, const double dir[3], const double pol[6], int comp, double k0,
                             double n_lo, double n_hi, int ncoarse, int nfine, double fine_step, double tol,
                             double out[6]);

/* The same retrieval for many lines at once - the three (direction, polarisation) pairs of a tensor, a
 * sweep over propagation directions at fixed omega (Fresnel normal surface), a frequency list
 * (k0 differs per line) - with ALL lines' points of a stage in ONE gsm_scan, so that the lock-step batch stays full.
 * dir[nlines][3] unit vectors, pol[nlines][6], comp[nlines] in {0, 1, 2} or -1 = projection of the 0-th order field on the
 * amplitude (sum_c conj(a_c) E_c / |a|^2, for off-axis directions), k0, n_lo, n_hi [nlines].  out[nlines][6] as
 * gsm_retrieve_neff (NaN for a line without a pole in its window); line_status[nlines] (may be NULL) GSM_OK or
 * GSM_E_INVALID per line.  Returns GSM_E_INVALID if any line failed, after filling the others. */
gsm_status gsm_retrieve_neff_many(gsm_plan* plan, int nlines, const double* dir, const double* pol, const int* comp,
                                  const double* k0, const double* n_lo, const double* n_hi, int ncoarse, int nfine,
                                  double fine_step, double tol, double* out, int* line_status);

/* ---- Operator apply for callers that cannot allocate -------------------------------------------------------------------
 * gsm_apply_static computes the same y[b] = x[b] - G(k_bloch[b], k0[b]) (T x[b]) as gsm_apply (Eq. 4; with
 * formulation = GSM_FORM_H the operator of Eq. 5), but takes no plan and calls no cudaMalloc, cudaFree,
 * cudaMallocHost or other allocating routine - not on the first call either.
 *
 * Who needs it: gsm_plan_create takes all of a plan's memory from cudaMalloc.  A program that embeds this library may be
 * unable to do that - its own allocator (a deep-learning framework's caching allocator, a server's pre-reserved pool)
 * already owns the device memory so that a further cudaMalloc fails or escapes its accounting, it runs under a per-client
 * memory quota, or it sits in a latency-bound loop where the device-wide synchronisation of cudaMalloc / cudaFree is not
 * acceptable.  Such a caller passes buffers from its own allocator for the inputs and the output; the intermediates
 * (transformed coefficient grid, z-transformed field) go to a fixed array of GSM_STATIC_SCRATCH_BYTES that is part of the
 * library image: every GPU that loads the library carries those bytes until the process exits, used or not.
 *
 * Limits (the price of a fixed array): orders[a] <= GSM_STATIC_MAX_ORDER per axis, batch <= GSM_STATIC_MAX_BATCH.  Anything
 * larger is refused with GSM_E_INVALID and a text from gsm_last_error(NULL) that names the limit; nothing is written.
 *
 * Arguments: period[3], orders[3], eps_b, formulation as in gsm_plan_desc.  d_coef: DEVICE, the Toeplitz generator c_d
 * ((2N1-1)(2N2-1)(2N3-1) complex, the layout of gsm_plan_coeffs; D_d for GSM_FORM_H), read on every call - the spectrum is
 * rebuilt each time since there is no plan to keep it.  k_bloch[batch][3], k0[batch]: HOST, copied before return.
 * d_x, d_y: DEVICE, [batch][3][N1][N2][N3] complex, 16-byte aligned, not overlapping.  cuda_stream: cudaStream_t to enqueue
 * on (NULL = legacy default stream).  All device pointers belong to the CURRENT device.  Asynchronous like gsm_apply.
 *
 * First call on a device: looks up the array's device address, sets kernel attributes and copies 1 KiB of FFT twiddles
 * into it with a synchronous cudaMemcpy.  Make that first call outside any stream capture.
 *
 * Sharing: there is ONE array per device.  Every call on that device uses it, and it keeps the previous call's contents;
 * the entry point clears or fully overwrites whatever it later reads, so stale contents never matter.  Calls that overlap
 * on the GPU (two streams, two host threads) race on the array and give wrong results - the caller must serialise them. */
#define GSM_STATIC_MAX_ORDER 16
#define GSM_STATIC_MAX_BATCH 4
#define GSM_STATIC_SCRATCH_BYTES 2622720
gsm_status gsm_apply_static(const double period[3], const int orders[3], double eps_b_re, double eps_b_im, int formulation,
                            const void* d_coef, int batch, const double* k_bloch, const double* k0, const void* d_x,
                            void* d_y, void* cuda_stream);

/* Text of the last failure on this plan (or, when plan == NULL, of the last failed gsm_plan_create or gsm_apply_static). */
const char* gsm_last_error(const gsm_plan* plan);

#ifdef __cplusplus
}
#endif
#endif /* GSM_H_ */
