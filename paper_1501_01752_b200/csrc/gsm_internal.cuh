// gsm_internal.cuh - shared declarations of the CUDA library behind include/gsm.h (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <vector>

#include "fft_device.cuh"
#include "gsm.h"

namespace gsm {

// Kernel classes for launch counting and (optional) per-class CUDA-event timing (gsm_plan_profile).
enum KernelClass {
    KC_Z_FORWARD = 0, KC_XY_CONV, KC_Z_INVERSE_GREEN, KC_SWEEP_DOTS, KC_HSOLVE, KC_SWEEP_UPDATE, KC_GIVENS,
    KC_NORMALIZE, KC_ARNOLDI_MGS, KC_COMBINE, KC_RESIDUAL, KC_SMALL, KC_PLAN, KC_APPLY_FUSED, KC_COUNT
};
const char* kernel_class_name(int cls);

// Counts every kernel launch per class; when `on`, also brackets each launch with a CUDA event pair on the launch
// stream (events are pooled and read back by collect()).
struct Profiler {
    bool on = false;
    long long launches[KC_COUNT] = {};
    double ms[KC_COUNT] = {};
    double bytes[KC_COUNT] = {};   // algorithmic bytes (minimal reads + writes of that kernel), summed over launches
    std::vector<cudaEvent_t> ev;   // pairs: ev[2i] start, ev[2i+1] stop
    std::vector<int> cls;
    size_t used = 0;
    void begin(int c, cudaStream_t st, double nbytes);
    void end(cudaStream_t st);
    cudaError_t collect();          // sync the events recorded so far and add their durations to ms[]
    void reset();
    void destroy();
};
struct ProfScope {
    Profiler* p; cudaStream_t st;
    ProfScope(Profiler* p_, int c, cudaStream_t st_, double nbytes = 0.0) : p(p_), st(st_) { if (p) p->begin(c, st, nbytes); }
    ~ProfScope() { if (p) p->end(st); }
};

// Geometry of the operator apply shared by the three passes.
struct ApplyGeom {
    AxisPlan ax[3];      // x, y, z axes of the circulant grid
    int N1, N2, N3;      // harmonics kept
    int NL;              // N1*N2 = number of z-lines per component
    long n;              // N1*N2*N3
    int hform;           // 0: Eq. 4 (E, Green dyadic); 1: Eq. 5 (H, cross products around the Toeplitz product)
    int L;               // z-lines per CTA in passes 1 and 3
    int Lst;             // odd row stride (>= L) of the pass-1 tile
    int RS3;             // odd row stride (>= 3L) of the pass-3 tile
    int N1s;             // odd row stride (>= N1) of the pass-2 plane
    int CB, CBs;         // columns per x-batch in pass 2 and the odd row stride (>= CB) of its scratch
    int split;           // 1: the xy plane does not fit shared memory (65..128 harmonics in x and y): pass 2 runs as
                         // y-expand -> x-convolution -> y-contract through the global workspace Y
    int YR, YRs;         // rows (i1) per CTA in the y passes of the split path and their odd stride
    cplx* Y;             // split path: [batch][3][P3][N1][P2], expanded along y only
    const cplx* tw[3];   // device twiddle tables exp(-2 pi i k / P_a)
    const cplx* chat;    // coefficient spectrum, position order, [P3][P1][P2], scaled by 1/(P1 P2 P3)
    const cplx* chat64;  // same, permuted for apply64.cu (null unless apply64_usable)
    const cplx* chat128; // same, in the order of apply128.cu's x/y network (null unless apply128_usable)
    double K[3];         // 2 pi / Lambda_a
    int mmin[3];         // lowest order per axis
    double epsb_re, epsb_im;
    // slot-refill scan (gsm_scan with more points than max_batch): solve b reads x and writes y at an extra offset of
    // jslot[b] * jstride complex numbers (its own Arnoldi index times the stride between basis vectors); null otherwise
    const int* jslot;
    long jstride;
};
// extra offset of solve b's x and y (see ApplyGeom.jslot)
static __device__ __forceinline__ long slot_offset(const ApplyGeom& g, int b) {
    return g.jslot ? (long)g.jslot[b] * g.jstride : 0L;
}

struct KrylovDims {
    long vlen;       // 3n complex numbers per vector
    int nchunk;      // CTAs per vector in the sweeps
    int chunk;       // elements per CTA (= threads * elems per thread)
    int mmax;        // max iterations (basis holds mmax+1 vectors)
    int ld;          // mmax + 1
    long vstride;    // complex numbers between consecutive basis vectors of one solve; 0 = batch * vlen (the kernels'
                     // `batch` argument); set when a launch covers only a group of the batch's solves
};
#define GSM_MAX_GROUPS 4   // sub-batches of one lock-step batch that iterate on streams of their own (gsm_api.cu run_batch)

// Device state of the fused persistent apply for 64-point axes (apply_fused64.cu); ring == null: not in use.
struct Fused64Dev {
    int* head = nullptr;        // [1] ticket counter
    int* cnt = nullptr;         // [3][maxB] per-solve completion counters of the three item kinds
    int* nact = nullptr;        // [1] number of listed solves
    int* list = nullptr;        // [maxB] batch indices of the solves of this launch
    const int* items = nullptr; // [items per slot] slot pattern
    cplx* ring = nullptr;       // W ring: [F64_RING][3][64][NL]
    int maxB = 0, grid = 0;     // counters' stride; persistent grid size (CTAs)
};

// ---- launches implemented in apply.cu --------------------------------------------------------------------------
// y[b] = x[b] - G_b (T x[b]); kvec[b][3], k0[b] device arrays; W workspace [batch][3][P3][NL] (three-launch path) or
// `fused` (one persistent launch, 64-point axes).  active (may be null): per-solve flags; solves with active[b] == 0
// are skipped.  units = number of solves whose algorithmic bytes are billed to the profiler now (run_batch bills the
// iteration loop afterwards from the final iteration counts and passes 0).
cudaError_t launch_apply(const ApplyGeom& g, int batch, const double* d_kvec, const double* d_k0, const cplx* d_x,
                         cplx* d_y, cplx* d_W, const Fused64Dev* fused, const int* d_active, cudaStream_t st,
                         Profiler* prof, double units);
// algorithmic bytes of `units` solve-applies (per-launch terms excluded) added to the apply's kernel classes
void bill_apply(const ApplyGeom& g, bool fused, Profiler* prof, double units);
// apply_fused64.cu
size_t fused64_ring_elems(const ApplyGeom& g);
int fused64_items_per_slot(const ApplyGeom& g);
void fused64_slot_pattern(const ApplyGeom& g, int* items);
cudaError_t apply_fused64_init_attributes(int* grid_out);
cudaError_t launch_apply_fused64(const ApplyGeom& g, int batch, const double* d_kvec, const double* d_k0, const cplx* d_x,
                                 cplx* d_y, const int* d_active, const Fused64Dev& f, cudaStream_t st);
size_t apply_smem_max(const ApplyGeom& g);
size_t apply_smem_plane(const ApplyGeom& g);   // shared memory of the single-kernel xy pass (decides ApplyGeom.split)
cudaError_t apply_init_attributes();
// apply128.cu: pass 2 specialised for 128-point x and y axes
bool apply128_usable(const ApplyGeom& g);
int apply128_freq_of_pos(int p);
cudaError_t apply128_init_attributes();
cudaError_t launch_chat128_layout(const cplx* d_chat, int P3, const int* d_gen1, const int* d_gen2, cplx* d_chat128,
                                  cudaStream_t st);
cudaError_t launch_xy_conv128(const ApplyGeom& g, int batch, cplx* d_W, const cplx* d_chat128, const int* d_active,
                              cudaStream_t st);
// apply64.cu: passes specialised for 64-point axes (chat64 = Chat permuted for 8-lane groups)
bool apply64_usable(const ApplyGeom& g);
cudaError_t apply64_init_attributes();
cudaError_t launch_chat64_layout(const cplx* d_chat, cplx* d_chat64, cudaStream_t st);
cudaError_t launch_z_forward64(const ApplyGeom& g, int batch, const cplx* d_x, cplx* d_W, const double* d_kvec,
                               const int* d_active, cudaStream_t st);
cudaError_t launch_z_inverse_green64(const ApplyGeom& g, int batch, const cplx* d_W, const cplx* d_x, cplx* d_y,
                                     const double* d_kvec, const double* d_k0, const int* d_active, cudaStream_t st);
cudaError_t launch_xy_conv64(const ApplyGeom& g, int batch, cplx* d_W, const cplx* d_chat64, const int* d_active,
                             cudaStream_t st);
cudaError_t plan_init_attributes();

// plan-time (a0): coefficients and their spectrum
struct ShapeDev {
    int kind;
    double c[3], s[3], dre, dim;  // centre, size, (eps_i - eps_bg)/eps_b
    double f;                     // volume fraction (polyhedron: 1 / cell volume, the image carries the volume)
    int f0, nf;                   // polyhedron: its faces in the PolyFace array
    double vol;                   // polyhedron: volume
};
// Polyhedron geometry prepared on the host: per face the outward unit normal, the area, one point of the face and its
// edges; per edge a -> b the midpoint, the half vector (b - a) / 2 and L m (length times in-plane outward normal).
struct PolyFace { double n[3], p0[3], area; int e0, ne; };
struct PolyEdge { double mid[3], half[3], mL[3]; };
cudaError_t launch_coeffs_analytic(const ShapeDev* d_shapes, int nshapes, const PolyFace* d_faces, const PolyEdge* d_edges,
                                   double c0_re, double c0_im, const double K[3], const int N[3], cplx* d_coef,
                                   cudaStream_t st);
// generic forward FFT along one axis of a dense [outer][P][inner] complex array in global memory (plan time only)
cudaError_t launch_fft_axis(cplx* d_data, long outer, const AxisPlan& ax, long inner, const cplx* d_tw, cudaStream_t st);
cudaError_t launch_embed(const cplx* d_coef, const int N[3], const int P[3], cplx* d_pad, cudaStream_t st);
cudaError_t launch_chat_layout(const cplx* d_padfft, const int P[3], cplx* d_chat, cudaStream_t st);
cudaError_t launch_voxel_prepare(cplx* d_grid, long count, double epsb_re, double epsb_im, int hform, cudaStream_t st);
// direct DFT of one axis of [outer][V][inner] keeping |d| <= N - 1: out[outer][2N-1][inner], scaled by 1 / V
cudaError_t launch_voxel_dft_axis(const cplx* d_in, long outer, int V, long inner, int N, cplx* d_out, cudaStream_t st);
cudaError_t launch_voxel_extract(const cplx* d_gridfft, const int Nv[3], const int N[3], const int* d_pos1,
                                 const int* d_pos2, const int* d_pos3, cplx* d_coef, cudaStream_t st);

// ---- launches implemented in krylov.cu -------------------------------------------------------------------------
struct KrylovState {   // all device pointers, one entry (or row) per solve of the batch
    cplx* basis;       // [ld][batch][vlen]
    cplx* part;        // [batch][2*ld][nchunk] partial inner products of sweep 1 / partial norms of sweep 2 (row 0)
    cplx* gram;        // [batch][ld][ld]   gram[j][i] = <v_i, v_j>, i <= j
    cplx* hcol;        // [batch][ld]       current Hessenberg column after Gram-Schmidt
    cplx* R;           // [batch][ld][mmax] rotated Hessenberg (upper triangular)
    double* cs;        // [batch][mmax]
    cplx* sn;          // [batch][mmax]
    cplx* g;           // [batch][ld]
    cplx* ycoef;       // [batch][mmax]
    double* hist;      // [batch][mmax]
    double* beta;      // [batch] ||r0||: norm of the first basis vector's unnormalised form
    double* bnorm;     // [batch] ||b||: the stop test and the reported residuals are relative to it
    int* guess;        // [batch] 1 when the solve starts from an initial guess x0 (r0 = b - A x0, x = x0 + d)
    int* rflag;        // [batch] 1 when the true residual needs one more apply (0: guess accepted as is, ||r0|| is it)
    double* scale;     // [batch] 1 / h_{j+1,j} of the running iteration
    int* active;       // [batch] 1 while iterating
    int* iters;        // [batch]
    int* nactive;      // [1]
    double* pol;       // [batch][6]
    double* tol;       // [1]
    // slot-refill scan only
    int* running;      // [batch] 1 while the slot holds a point whose results have not been recorded yet
    int* fin;          // [batch] solve finished in this tick: 1 converged, 2 stopped at max_iters
    int* point;        // [batch] list index of the slot's point
    int* newv;         // [batch] slot was handed a new point in this tick
};
// Device side of a slot-refill scan: the whole point list and the per-point outputs.
struct RefillDev {
    const double* kvec_all;   // [npts][3]
    const double* k0_all;     // [npts]
    const double* pol_all;    // [npts][6]
    int npts;
    int* next;                // [1] first point not handed out yet
    int* ndone;               // [1] points whose results are recorded
    int* out_iters;           // [npts]
    double* out_resid;        // [npts]
    cplx* out_resp;           // [npts][3]
    int* out_flag;            // [npts] 1: stopped at max_iters
};
// view of the per-solve state that starts at solve b0 (every array advanced by b0 entries / rows); nactive = counter
KrylovState krylov_state_view(const KrylovDims& d, const KrylovState& s, int b0, int* nactive);
// counts[g] = number of active solves in [bounds[g], bounds[g + 1]), g < ngroups <= GSM_MAX_GROUPS
struct GroupBounds { int b[GSM_MAX_GROUPS + 1]; };
cudaError_t launch_group_count(const KrylovState& s, int ngroups, GroupBounds bounds, int* d_counts, cudaStream_t st, Profiler* prof);
cudaError_t launch_krylov_init(const KrylovDims& d, const KrylovState& s, int batch, long i0 /*index of m=0*/, long n,
                               cudaStream_t st, Profiler* prof);
cudaError_t launch_sweep_dots(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof);
cudaError_t launch_hsolve(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof);
cudaError_t launch_sweep_update(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof);
cudaError_t launch_givens(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof);
cudaError_t launch_normalize(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof);
// d_mask (may be null): per-solve flags, solves with mask[b] == 0 are skipped (also in launch_combine / launch_mesh_scatter)
cudaError_t launch_backsolve(const KrylovDims& d, const KrylovState& s, int batch, cudaStream_t st, Profiler* prof,
                             const int* d_mask = nullptr);
// E[b] = (guess[b] ? x0[b] : 0) + sum_i y_i v_i; x0 may be null and may alias d_E
cudaError_t launch_combine(const KrylovDims& d, const KrylovState& s, int batch, const cplx* d_x0, cplx* d_E, cudaStream_t st,
                           Profiler* prof, const int* d_mask = nullptr);
// Start from an initial guess (Saad Alg. 6.9 with x0 != 0): given y = A x0 in basis slot 1, set
// r0 = b - y, beta = ||r0||, v_0 = r0 / beta, g_0 = beta for every solve whose guess beats the zero start
// (||r0|| < ||b||); the others keep the state launch_krylov_init gave them.
cudaError_t launch_krylov_guess(const KrylovDims& d, const KrylovState& s, int batch, long i0, long n, cudaStream_t st,
                                Profiler* prof);
// scan over an ordered mesh (gsm_scan_mesh): guesses by interpolation of already solved neighbours, and the scatter
// of a wave's solutions into the mesh-ordered field array.  nbr[b][GSM_MESH_NNB] = neighbour point indices (-1: unused),
// wgt[b][GSM_MESH_NNB] their (complex) weights, idx[b] = point index of solve b.
#ifndef GSM_MESH_NNB
#define GSM_MESH_NNB 8   // interpolation nodes per guess: the solved neighbours at distance s, 3 s, 5 s, 7 s on both sides
                         // (measured on the bench workload, ms per 256-point scan: 4 nodes 30.2, 6 nodes 20.9, 8 nodes 19.0)
#endif
cudaError_t launch_mesh_guess(const KrylovDims& d, int batch, const cplx* d_all, const int* d_nbr, const cplx* d_wgt,
                              cplx* d_x0, cudaStream_t st, Profiler* prof);
cudaError_t launch_mesh_scatter(const KrylovDims& d, int batch, const cplx* d_src, const int* d_idx, cplx* d_all,
                                cudaStream_t st, Profiler* prof, const int* d_mask = nullptr);
// slot-refill scan: mark the solves that finished in this tick; record their results and hand out the next points
cudaError_t launch_refill_mark(const KrylovDims& d, const KrylovState& s, int batch, cudaStream_t st, Profiler* prof);
cudaError_t launch_refill_commit(const KrylovDims& d, const KrylovState& s, const RefillDev& r, int batch, long i0, long n,
                                 const cplx* d_E_slot, const double* d_resid_slot, double* d_kvec_slot, double* d_k0_slot,
                                 cudaStream_t st, Profiler* prof);
// rflag[b] = 0 for the solves whose guess met the stop test without iterating (E = x0 and the true residual is the
// ||r0|| / ||b|| already formed from A x0), 1 for all others
cudaError_t launch_residual_select(const KrylovDims& d, const KrylovState& s, int batch, cudaStream_t st, Profiler* prof);
// resid[b] = || pol delta_m0 - y[b] || / ||b|| where rflag[b] != 0 (y = A E from one more apply), else ||r0|| / ||b||
cudaError_t launch_true_residual(const KrylovDims& d, const KrylovState& s, int batch, const cplx* d_y, long i0, long n,
                                 double* d_resid, cudaStream_t st, Profiler* prof);
cudaError_t krylov_init_attributes();

// ---- launches implemented in arnoldi_cluster.cu ------------------------------------------------------------------
// One Arnoldi step (MGS + norm + normalise + Givens) per solve in one thread-block cluster, basis read once.
// arnoldi_cluster_plan: cluster size (0 = not usable: fall back to the two-sweep kernels) and elements per CTA.
cudaError_t arnoldi_cluster_plan(const KrylovDims& d, int* cs_out, int* chunk_out, int* nclusters_out);
cudaError_t launch_arnoldi_cluster(const KrylovDims& d, const KrylovState& s, int batch, int j, int cs, int chunk,
                                   int nclusters, cudaStream_t st, Profiler* prof);

}  // namespace gsm
