// gsm_api.cu - the C ABI of include/gsm.h: plan construction, operator apply, batched GMRES solve and scan.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>
#include <utility>

#include "gsm_internal.cuh"

using namespace gsm;

static thread_local std::string g_create_error;

struct gsm_plan {
    gsm_plan_desc desc{};
    ApplyGeom geom{};
    KrylovDims kd{};
    KrylovState ks{};
    cudaStream_t stream = nullptr;
    int max_batch = 1, max_iters = 64;
    int last_nb = 0;              // size of the most recent lock-step batch (gsm_plan_history)
    long i0 = 0;                  // flat index of m = 0 inside one component
    int mgs_cs = 0, mgs_chunk = 0, mgs_nclusters = 0; // cluster MGS Arnoldi step (0 = two-sweep fallback)
    Fused64Dev fused;             // fused persistent apply for 64-point axes (ring == null: three-launch apply)
    std::vector<void*> allocs;    // every device allocation, freed in destroy
    long long device_bytes = 0;
    Profiler prof;
    cudaEvent_t iter_ev[2] = {nullptr, nullptr};   // completion of the per-iteration nactive read-back
    // groups of one lock-step batch iterating concurrently (run_batch): group 0 on `stream`, the others on streams of their own
    cudaStream_t gstream[GSM_MAX_GROUPS] = {};
    cudaEvent_t gev[GSM_MAX_GROUPS][2] = {};       // per-group read-back events
    cudaEvent_t gsync[GSM_MAX_GROUPS] = {};        // fork ([0]) / join
    int* d_gcount = nullptr;                       // [GSM_MAX_GROUPS] solves of each group still iterating

    cplx* chat64 = nullptr;
    cplx* chat128 = nullptr;
    int* gen128[2] = {nullptr, nullptr};
    cplx *coef = nullptr, *chat = nullptr, *pad = nullptr, *W = nullptr, *xbuf = nullptr, *ybuf = nullptr;
    size_t vgrid_count = 0;
    cplx* vgrid = nullptr;        // voxel path: device copy of the grid, transformed in place
    const cplx* vtw[3] = {nullptr, nullptr, nullptr};
    int* vpos[3] = {nullptr, nullptr, nullptr};
    int vdim[3] = {0, 0, 0};
    double *d_kvec = nullptr, *d_k0 = nullptr, *d_resid = nullptr;
    cplx* mesh_fields = nullptr;  // gsm_scan_mesh without d_E_out: every solution of the mesh (grown on demand)
    size_t mesh_cap = 0;
    int *d_mesh_idx = nullptr, *d_mesh_nbr = nullptr;   // [max_batch], [max_batch][4]
    cplx* d_mesh_wgt = nullptr;                         // [max_batch][4]
    void* refill_buf = nullptr;   // slot-refill scan: point list and per-point outputs on the device (grown on demand)
    size_t refill_cap = 0;        // points it holds
    int* d_refill_ctl = nullptr;  // [2] next point, points done
    void* pinned = nullptr;       // host staging: nactive, iters, resid, hist
    size_t pinned_bytes = 0;
    mutable std::string err;
};

#define CK(call)                                                                                      \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess) {                                                                      \
            char buf_[512];                                                                           \
            snprintf(buf_, sizeof buf_, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return fail(plan, e_ == cudaErrorMemoryAllocation ? GSM_E_ALLOC : GSM_E_CUDA, buf_);       \
        }                                                                                             \
    } while (0)

static gsm_status fail(const gsm_plan* plan, gsm_status st, const char* msg) {
    if (plan) plan->err = msg; else g_create_error = msg;
    return st;
}

template <typename T>
static cudaError_t dalloc(gsm_plan* p, T** out, size_t count) {
    void* q = nullptr;
    const size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
    cudaError_t e = cudaMalloc(&q, bytes);
    if (e != cudaSuccess) return e;
    p->allocs.push_back(q);
    p->device_bytes += (long long)bytes;
    *out = static_cast<T*>(q);
    return cudaSuccess;
}

// Give back one block obtained from dalloc (used where a workspace is replaced by one of another size).
template <typename T>
static void dfree(gsm_plan* p, T** ptr, size_t count) {
    if (!*ptr) return;
    auto it = std::find(p->allocs.begin(), p->allocs.end(), static_cast<void*>(*ptr));
    if (it != p->allocs.end()) p->allocs.erase(it);
    cudaFree(*ptr);
    p->device_bytes -= (long long)(std::max<size_t>(count, 1) * sizeof(T));
    *ptr = nullptr;
}

static int fft_size(int N) {
    if (N == 1) return 1;
    int p = 1;
    while (p < 2 * N - 1) p *= 2;
    return p;
}

// radix plan of a power-of-two length (fft_device.cuh): larger radices last, so the fused middle stage is wide
static bool make_axis(int P, int N, AxisPlan* ax) {
    ax->P = P; ax->N = N; ax->nst = 0;
    for (int i = 0; i < 4; ++i) ax->radix[i] = 1;
    switch (P) {
        case 1: break;
        case 2: ax->nst = 1; ax->radix[0] = 2; break;
        case 4: ax->nst = 1; ax->radix[0] = 4; break;
        case 8: ax->nst = 1; ax->radix[0] = 8; break;
        case 16: ax->nst = 2; ax->radix[0] = 4; ax->radix[1] = 4; break;
        case 32: ax->nst = 2; ax->radix[0] = 4; ax->radix[1] = 8; break;
        case 64: ax->nst = 2; ax->radix[0] = 8; ax->radix[1] = 8; break;
        case 128: ax->nst = 3; ax->radix[0] = 4; ax->radix[1] = 4; ax->radix[2] = 8; break;
        case 256: ax->nst = 3; ax->radix[0] = 4; ax->radix[1] = 8; ax->radix[2] = 8; break;
        case 512: ax->nst = 3; ax->radix[0] = 8; ax->radix[1] = 8; ax->radix[2] = 8; break;
        default: return false;
    }
    return true;
}

// position (after the forward network) of frequency k: q = k mod R0 selects block q, the rest recurses
static int pos_of_freq(int k, int P, const int* radix, int nst) {
    int pos = 0;
    for (int s = 0; s < nst; ++s) {
        const int R = radix[s];
        P /= R;
        pos += (k % R) * P;
        k /= R;
    }
    return pos;
}

static cudaError_t upload_twiddles(gsm_plan* p, int P, const cplx** out) {
    std::vector<double> h(2 * (size_t)P);
    for (int k = 0; k < P; ++k) {
        const double a = -2.0 * M_PI * (double)k / (double)P;
        h[2 * k] = std::cos(a);
        h[2 * k + 1] = std::sin(a);
    }
    // exact values on the axes
    if (P >= 2) { h[2 * (P / 2)] = -1.0; h[2 * (P / 2) + 1] = 0.0; }
    if (P >= 4) { h[2 * (P / 4)] = 0.0; h[2 * (P / 4) + 1] = -1.0; h[2 * (3 * P / 4)] = 0.0; h[2 * (3 * P / 4) + 1] = 1.0; }
    cplx* d = nullptr;
    cudaError_t e = dalloc(p, &d, (size_t)P);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(d, h.data(), sizeof(double) * 2 * P, cudaMemcpyHostToDevice);
    *out = d;
    return e;
}

static int odd_at_least(int v) { return v | 1; }

static cplx cdivh(double ar, double ai, double br, double bi) {
    const double inv = 1.0 / (br * br + bi * bi);
    return make_double2((ar * br + ai * bi) * inv, (ai * br - ar * bi) * inv);
}

// Polyhedron geometry for the device (plan_kernels.cu polyhedron_image): normals, areas, edges.  Returns null, or the
// reason the description is malformed: index out of range, degenerate or non-planar face, fewer than 4 faces, a surface
// that is not closed and consistently oriented (every directed edge a -> b of a face must be matched by exactly one
// b -> a of another face: one face listed clockwise, a missing face or a doubled face all break this), or inward
// orientation as a whole (negative volume).  The closed form of reading R27 is only valid for such a surface.
static const char* prepare_polyhedron(const gsm_shape& s, ShapeDev& q, std::vector<PolyFace>& faces, std::vector<PolyEdge>& edges) {
    if (s.n_vertices < 4 || s.n_faces < 4 || !s.vertices || !s.face_sizes || !s.face_vertices)
        return "polyhedron needs at least 4 vertices and 4 faces";
    std::map<std::pair<int, int>, int> directed;   // directed edge -> how often it occurs
    q.f0 = (int)faces.size();
    q.nf = s.n_faces;
    q.vol = 0.0;
    const int* fv = s.face_vertices;
    for (int f = 0; f < s.n_faces; ++f) {
        const int cnt = s.face_sizes[f];
        if (cnt < 3) return "polyhedron face with fewer than 3 vertices";
        for (int k = 0; k < cnt; ++k)
            if (fv[k] < 0 || fv[k] >= s.n_vertices) return "polyhedron vertex index out of range";
        for (int k = 0; k < cnt; ++k) {
            const int a = fv[k], b = fv[(k + 1) % cnt];
            if (a == b || ++directed[std::make_pair(a, b)] > 1) return "polyhedron surface is not closed and consistently oriented (repeated edge)";
        }
        auto V = [&](int k) { return s.vertices + 3 * (size_t)fv[k % cnt]; };
        PolyFace F{};
        double nv[3] = {0.0, 0.0, 0.0};
        for (int k = 1; k + 1 < cnt; ++k) {           // area vector of the fan triangulation
            const double a[3] = {V(k)[0] - V(0)[0], V(k)[1] - V(0)[1], V(k)[2] - V(0)[2]};
            const double b[3] = {V(k + 1)[0] - V(0)[0], V(k + 1)[1] - V(0)[1], V(k + 1)[2] - V(0)[2]};
            nv[0] += 0.5 * (a[1] * b[2] - a[2] * b[1]);
            nv[1] += 0.5 * (a[2] * b[0] - a[0] * b[2]);
            nv[2] += 0.5 * (a[0] * b[1] - a[1] * b[0]);
        }
        F.area = std::sqrt(nv[0] * nv[0] + nv[1] * nv[1] + nv[2] * nv[2]);
        if (!(F.area > 0.0)) return "degenerate polyhedron face (zero area)";
        for (int a = 0; a < 3; ++a) { F.n[a] = nv[a] / F.area; F.p0[a] = V(0)[a]; }
        for (int k = 1; k < cnt; ++k) {               // planarity: distance of every vertex from the plane through V(0)
            const double dist = (V(k)[0] - F.p0[0]) * F.n[0] + (V(k)[1] - F.p0[1]) * F.n[1] + (V(k)[2] - F.p0[2]) * F.n[2];
            if (std::fabs(dist) > 1e-9 * std::sqrt(F.area)) return "polyhedron face is not planar";
        }
        q.vol += (F.p0[0] * F.n[0] + F.p0[1] * F.n[1] + F.p0[2] * F.n[2]) * F.area / 3.0;
        F.e0 = (int)edges.size();
        F.ne = cnt;
        for (int k = 0; k < cnt; ++k) {
            PolyEdge E{};
            double d[3];
            for (int a = 0; a < 3; ++a) {
                d[a] = V(k + 1)[a] - V(k)[a];
                E.mid[a] = 0.5 * (V(k + 1)[a] + V(k)[a]);
                E.half[a] = 0.5 * d[a];
            }
            // L m = L (t x n) = (b - a) x n
            E.mL[0] = d[1] * F.n[2] - d[2] * F.n[1];
            E.mL[1] = d[2] * F.n[0] - d[0] * F.n[2];
            E.mL[2] = d[0] * F.n[1] - d[1] * F.n[0];
            edges.push_back(E);
        }
        faces.push_back(F);
        fv += cnt;
    }
    for (const auto& kv : directed)
        if (!directed.count(std::make_pair(kv.first.second, kv.first.first)))
            return "polyhedron surface is not closed and consistently oriented (an edge without its reverse: open surface or a face listed clockwise)";
    return q.vol > 0.0 ? nullptr : "polyhedron faces are oriented inwards (list them counter-clockwise seen from outside)";
}

// voxel grid sizes: at least the 2N - 1 harmonics needed per axis (1 is allowed for an axis with one order)
static bool voxel_dims_ok(const int* V, const int* N) {
    for (int a = 0; a < 3; ++a)
        if (V[a] < 2 * N[a] - 1 || V[a] > 2048) return false;
    return true;
}

// a0: coefficients c_d on the device, either from closed forms or from a transform of the voxel grid
static gsm_status build_coeffs(gsm_plan* plan) {
    const gsm_plan_desc& d = plan->desc;
    const int* N = d.orders;
    const size_t ncoef = (size_t)(2 * N[0] - 1) * (2 * N[1] - 1) * (2 * N[2] - 1);
    if (!plan->coef) CK(dalloc(plan, &plan->coef, ncoef));
    if (d.eps_grid_host == nullptr) {
        std::vector<ShapeDev> hs(std::max(d.n_shapes, 1));
        std::vector<PolyFace> pfaces;
        std::vector<PolyEdge> pedges;
        const double vol = d.period[0] * d.period[1] * d.period[2];
        for (int i = 0; i < d.n_shapes; ++i) {
            const gsm_shape& s = d.shapes[i];
            ShapeDev& q = hs[i];
            q.kind = s.kind;
            for (int a = 0; a < 3; ++a) { q.c[a] = s.center[a]; q.s[a] = s.size[a]; }
            cplx del = cdivh(s.eps_re - d.eps_bg_re, s.eps_im - d.eps_bg_im, d.eps_b_re, d.eps_b_im);
            if (d.formulation == GSM_FORM_H) {   // eps_b/eps_bg - eps_b/eps_i
                const cplx a = cdivh(d.eps_b_re, d.eps_b_im, d.eps_bg_re, d.eps_bg_im);
                const cplx b = cdivh(d.eps_b_re, d.eps_b_im, s.eps_re, s.eps_im);
                del = make_double2(a.x - b.x, a.y - b.y);
            }
            q.dre = del.x; q.dim = del.y;
            if (s.kind == GSM_SPHERE) q.f = 4.0 / 3.0 * M_PI * s.size[0] * s.size[0] * s.size[0] / vol;
            else if (s.kind == GSM_ELLIPSOID) q.f = 4.0 / 3.0 * M_PI * s.size[0] * s.size[1] * s.size[2] / vol;
            else if (s.kind == GSM_BOX) q.f = s.size[0] * s.size[1] * s.size[2] / vol;
            else if (s.kind == GSM_POLYHEDRON) {
                q.f = 1.0 / vol;
                if (const char* why = prepare_polyhedron(s, q, pfaces, pedges)) return fail(plan, GSM_E_INVALID, why);
            } else return fail(plan, GSM_E_INVALID, "unknown shape kind");
        }
        ShapeDev* dsh = nullptr;
        PolyFace* dfaces = nullptr;
        PolyEdge* dedges = nullptr;
        CK(cudaMalloc(&dsh, sizeof(ShapeDev) * hs.size()));
        cudaError_t e = cudaMemcpyAsync(dsh, hs.data(), sizeof(ShapeDev) * hs.size(), cudaMemcpyHostToDevice, plan->stream);
        if (e == cudaSuccess && !pfaces.empty()) {
            e = cudaMalloc(&dfaces, sizeof(PolyFace) * pfaces.size());
            if (e == cudaSuccess) e = cudaMalloc(&dedges, sizeof(PolyEdge) * pedges.size());
            if (e == cudaSuccess) e = cudaMemcpyAsync(dfaces, pfaces.data(), sizeof(PolyFace) * pfaces.size(), cudaMemcpyHostToDevice, plan->stream);
            if (e == cudaSuccess) e = cudaMemcpyAsync(dedges, pedges.data(), sizeof(PolyEdge) * pedges.size(), cudaMemcpyHostToDevice, plan->stream);
        }
        cplx c0 = cdivh(d.eps_bg_re - d.eps_b_re, d.eps_bg_im - d.eps_b_im, d.eps_b_re, d.eps_b_im);
        if (d.formulation == GSM_FORM_H)     // 1 - eps_b/eps_bg = (eps_bg - eps_b)/eps_bg
            c0 = cdivh(d.eps_bg_re - d.eps_b_re, d.eps_bg_im - d.eps_b_im, d.eps_bg_re, d.eps_bg_im);
        if (e == cudaSuccess) {
            ProfScope ps_(&plan->prof, KC_PLAN, plan->stream);
            e = launch_coeffs_analytic(dsh, d.n_shapes, dfaces, dedges, c0.x, c0.y, plan->geom.K, N, plan->coef, plan->stream);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(plan->stream);
        cudaFree(dsh);
        if (dfaces) cudaFree(dfaces);
        if (dedges) cudaFree(dedges);
        CK(e);
        return GSM_OK;
    }
    // voxel path: transform of (eps - eps_b)/eps_b on the Nv grid, keep |d_a| <= N_a - 1
    const int* V = d.voxels;
    if (!voxel_dims_ok(V, N)) return fail(plan, GSM_E_INVALID, "voxels[a] must satisfy 2N-1 <= voxels <= 2048");
    AxisPlan vax[3];
    bool pow2 = true;
    for (int a = 0; a < 3; ++a) pow2 = pow2 && V[a] <= 512 && make_axis(V[a], V[a], &vax[a]);
    if (!pow2) {   // any other size: the defining sums, axis by axis, each pass keeping only the wanted harmonics
        const size_t nv = (size_t)V[0] * V[1] * V[2];
        const size_t n1 = (size_t)V[0] * V[1] * (2 * N[2] - 1), n2 = (size_t)V[0] * (2 * N[1] - 1) * (2 * N[2] - 1);
        if (!plan->vgrid || plan->vgrid_count != nv + n1 + n2) {   // a grid of another size replaces the old block
            CK(cudaStreamSynchronize(plan->stream));
            dfree(plan, &plan->vgrid, plan->vgrid_count);
            plan->vgrid_count = 0;
            CK(dalloc(plan, &plan->vgrid, nv + n1 + n2));
            plan->vgrid_count = nv + n1 + n2;
        }
        cplx *grid = plan->vgrid, *t1 = grid + nv, *t2 = t1 + n1;
        cudaError_t e = cudaMemcpyAsync(grid, d.eps_grid_host, sizeof(cplx) * nv, cudaMemcpyHostToDevice, plan->stream);
        ProfScope ps_(&plan->prof, KC_PLAN, plan->stream);
        if (e == cudaSuccess) e = launch_voxel_prepare(grid, (long)nv, d.eps_b_re, d.eps_b_im, d.formulation == GSM_FORM_H, plan->stream);
        if (e == cudaSuccess) e = launch_voxel_dft_axis(grid, (long)V[0] * V[1], V[2], 1, N[2], t1, plan->stream);
        if (e == cudaSuccess) e = launch_voxel_dft_axis(t1, (long)V[0], V[1], 2 * N[2] - 1, N[1], t2, plan->stream);
        if (e == cudaSuccess) e = launch_voxel_dft_axis(t2, 1, V[0], (long)(2 * N[1] - 1) * (2 * N[2] - 1), N[0], plan->coef, plan->stream);
        CK(e);
        return GSM_OK;
    }
    if (!plan->vtw[0] || plan->vdim[0] != V[0] || plan->vdim[1] != V[1] || plan->vdim[2] != V[2]) {
        for (int a = 0; a < 3; ++a) {   // twiddles and frequency->position tables of the voxel FFT (kept for re-use)
            CK(upload_twiddles(plan, V[a], &plan->vtw[a]));
            std::vector<int> pos(V[a]);
            for (int k = 0; k < V[a]; ++k) pos[k] = pos_of_freq(k, V[a], vax[a].radix, vax[a].nst);
            CK(dalloc(plan, &plan->vpos[a], (size_t)V[a]));
            CK(cudaMemcpy(plan->vpos[a], pos.data(), sizeof(int) * V[a], cudaMemcpyHostToDevice));
            plan->vdim[a] = V[a];
        }
    }
    const cplx* const* vtw = plan->vtw;
    int* const* dpos = plan->vpos;
    const size_t nv = (size_t)V[0] * V[1] * V[2];
    if (!plan->vgrid || plan->vgrid_count != nv) {
        CK(cudaStreamSynchronize(plan->stream));
        dfree(plan, &plan->vgrid, plan->vgrid_count);
        plan->vgrid_count = 0;
        CK(dalloc(plan, &plan->vgrid, nv));
        plan->vgrid_count = nv;
    }
    cplx* grid = plan->vgrid;
    cudaError_t e = cudaMemcpyAsync(grid, d.eps_grid_host, sizeof(cplx) * nv, cudaMemcpyHostToDevice, plan->stream);
    ProfScope ps_(&plan->prof, KC_PLAN, plan->stream);
    if (e == cudaSuccess) e = launch_voxel_prepare(grid, (long)nv, d.eps_b_re, d.eps_b_im, d.formulation == GSM_FORM_H, plan->stream);
    if (e == cudaSuccess) e = launch_fft_axis(grid, (long)V[0] * V[1], vax[2], 1, vtw[2], plan->stream);
    if (e == cudaSuccess) e = launch_fft_axis(grid, (long)V[0], vax[1], V[2], vtw[1], plan->stream);
    if (e == cudaSuccess) e = launch_fft_axis(grid, 1, vax[0], (long)V[1] * V[2], vtw[0], plan->stream);
    if (e == cudaSuccess) e = launch_voxel_extract(grid, V, N, dpos[0], dpos[1], dpos[2], plan->coef, plan->stream);
    CK(e);
    return GSM_OK;
}

// Chat = forward network applied to the circulant embedding of c, laid out [pos3][pos1][pos2], scaled 1/(P1P2P3)
static gsm_status build_spectrum(gsm_plan* plan) {
    ApplyGeom& g = plan->geom;
    const int P[3] = {g.ax[0].P, g.ax[1].P, g.ax[2].P};
    const int N[3] = {g.N1, g.N2, g.N3};
    const size_t np = (size_t)P[0] * P[1] * P[2];
    if (!plan->chat) CK(dalloc(plan, &plan->chat, np));
    if (!plan->pad) CK(dalloc(plan, &plan->pad, np));
    cplx* pad = plan->pad;
    ProfScope ps_(&plan->prof, KC_PLAN, plan->stream);
    cudaError_t e = launch_embed(plan->coef, N, P, pad, plan->stream);
    AxisPlan full[3] = {g.ax[0], g.ax[1], g.ax[2]};
    if (e == cudaSuccess) e = launch_fft_axis(pad, (long)P[0] * P[1], full[2], 1, g.tw[2], plan->stream);
    if (e == cudaSuccess) e = launch_fft_axis(pad, (long)P[0], full[1], P[2], g.tw[1], plan->stream);
    if (e == cudaSuccess) e = launch_fft_axis(pad, 1, full[0], (long)P[1] * P[2], g.tw[0], plan->stream);
    if (e == cudaSuccess) e = launch_chat_layout(pad, P, plan->chat, plan->stream);
    const bool generic = (plan->desc.flags & GSM_FLAG_GENERIC_APPLY) != 0;
    if (e == cudaSuccess && apply64_usable(g) && !generic) {
        if (!plan->chat64) CK(dalloc(plan, &plan->chat64, np));
        e = launch_chat64_layout(plan->chat, plan->chat64, plan->stream);
        g.chat64 = plan->chat64;
    }
    if (e == cudaSuccess && apply128_usable(g) && !generic) {
        if (!plan->chat128) {
            CK(dalloc(plan, &plan->chat128, np));
            for (int a = 0; a < 2; ++a) {   // new position -> frequency -> position in the generic network
                std::vector<int> gen(128);
                for (int q = 0; q < 128; ++q) gen[q] = pos_of_freq(apply128_freq_of_pos(q), 128, g.ax[a].radix, g.ax[a].nst);
                CK(dalloc(plan, &plan->gen128[a], (size_t)128));
                CK(cudaMemcpy(plan->gen128[a], gen.data(), sizeof(int) * 128, cudaMemcpyHostToDevice));
            }
        }
        e = launch_chat128_layout(plan->chat, P[2], plan->gen128[0], plan->gen128[1], plan->chat128, plan->stream);
        g.chat128 = plan->chat128;
    }
    CK(e);
    g.chat = plan->chat;
    return GSM_OK;
}

extern "C" gsm_status gsm_plan_create(const gsm_plan_desc* desc, gsm_plan** out) {
    if (out) *out = nullptr;
    if (!desc || !out) return fail(nullptr, GSM_E_INVALID, "null descriptor or output pointer");
    for (int a = 0; a < 3; ++a) {
        if (desc->orders[a] < 1 || desc->orders[a] > 256) return fail(nullptr, GSM_E_INVALID, "orders must be in [1, 256]");
        if (!(desc->period[a] > 0.0)) return fail(nullptr, GSM_E_INVALID, "periods must be positive");
    }
    if (desc->eps_b_re == 0.0 && desc->eps_b_im == 0.0) return fail(nullptr, GSM_E_INVALID, "eps_b must be non-zero");
    if (desc->eps_grid_host == nullptr && (desc->n_shapes < 0 || (desc->n_shapes > 0 && !desc->shapes)))
        return fail(nullptr, GSM_E_INVALID, "shapes missing");
    // the two-sweep kernels stage (j + 1)-sized rows in shared memory and the pool holds max_iters + 1 vectors per solve
    if (desc->max_iters > GSM_MAX_ITERS) return fail(nullptr, GSM_E_INVALID, "max_iters exceeds GSM_MAX_ITERS");
    if (desc->flags & ~(GSM_FLAG_TWO_SWEEP | GSM_FLAG_GENERIC_APPLY | GSM_FLAG_FUSED_APPLY | GSM_FLAG_SLOT_REFILL))
        return fail(nullptr, GSM_E_INVALID, "unknown flag");
    gsm_plan* plan = new (std::nothrow) gsm_plan();
    if (!plan) return fail(nullptr, GSM_E_ALLOC, "host allocation failed");
    plan->desc = *desc;
    plan->stream = static_cast<cudaStream_t>(desc->cuda_stream);
    plan->max_batch = desc->max_batch > 0 ? desc->max_batch : 1;
    plan->max_iters = desc->max_iters > 0 ? desc->max_iters : 64;
    gsm_status st = GSM_OK;
    auto body = [&]() -> gsm_status {
        ApplyGeom& g = plan->geom;
        const int* N = desc->orders;
        g.N1 = N[0]; g.N2 = N[1]; g.N3 = N[2];
        g.NL = N[0] * N[1];
        g.n = (long)N[0] * N[1] * N[2];
        for (int a = 0; a < 3; ++a) {
            if (!make_axis(fft_size(N[a]), N[a], &g.ax[a])) return fail(plan, GSM_E_INVALID, "unsupported FFT size");
            g.K[a] = 2.0 * M_PI / desc->period[a];
            g.mmin[a] = (N[a] % 2 == 1) ? -(N[a] - 1) / 2 : -N[a] / 2;
            CK(upload_twiddles(plan, g.ax[a].P, &g.tw[a]));
        }
        g.epsb_re = desc->eps_b_re; g.epsb_im = desc->eps_b_im;
        if (desc->formulation != GSM_FORM_E && desc->formulation != GSM_FORM_H)
            return fail(plan, GSM_E_INVALID, "formulation must be GSM_FORM_E or GSM_FORM_H");
        g.hform = desc->formulation == GSM_FORM_H;
        g.L = std::min(g.NL, g.ax[2].P >= 512 ? 8 : g.ax[2].P >= 128 ? 16 : 32);
        g.Lst = odd_at_least(g.L);
        g.RS3 = odd_at_least(3 * g.L);
        g.N1s = odd_at_least(g.N1);
        g.CB = std::min(g.ax[1].P, g.ax[0].P >= 128 ? 16 : 32);
        g.CBs = odd_at_least(g.CB);
        g.YR = std::min(g.N1, g.ax[1].P >= 128 ? 16 : 32);
        g.YRs = odd_at_least(g.YR);
        // 65..128 harmonics in x and y: the pruned plane no longer fits one SM's shared memory
        g.split = apply_smem_plane(g) > 227 * 1024;
        if (apply_smem_max(g) > 227 * 1024) return fail(plan, GSM_E_INVALID, "orders too large for the shared-memory tiles");
        plan->i0 = ((long)(-g.mmin[0]) * N[1] + (-g.mmin[1])) * N[2] + (-g.mmin[2]);
        CK(apply_init_attributes());
        CK(plan_init_attributes());
        CK(krylov_init_attributes());
        gsm_status s2 = build_coeffs(plan);
        if (s2 != GSM_OK) return s2;
        s2 = build_spectrum(plan);
        if (s2 != GSM_OK) return s2;
        CK(cudaStreamSynchronize(plan->stream));
        // workspaces
        const int B = plan->max_batch, m = plan->max_iters;
        KrylovDims& kd = plan->kd;
        kd.vlen = 3 * g.n;
        kd.chunk = 256 * 4;
        kd.nchunk = (int)((kd.vlen + kd.chunk - 1) / kd.chunk);
        kd.mmax = m;
        kd.ld = m + 1;
        KrylovState& ks = plan->ks;
        CK(arnoldi_cluster_plan(kd, &plan->mgs_cs, &plan->mgs_chunk, &plan->mgs_nclusters));
        if (desc->flags & GSM_FLAG_TWO_SWEEP) plan->mgs_cs = 0;
        if (g.chat64 && (desc->flags & GSM_FLAG_FUSED_APPLY)) {
            // fused persistent apply: W lives in a ring of a few solve slots that stays in L2 (apply_fused64.cu)
            Fused64Dev& f = plan->fused;
            CK(apply_fused64_init_attributes(&f.grid));
            f.maxB = B;
            int* items = nullptr;
            const int ips = fused64_items_per_slot(g);
            std::vector<int> pattern(ips);
            fused64_slot_pattern(g, pattern.data());
            CK(dalloc(plan, &items, (size_t)ips));
            CK(cudaMemcpy(items, pattern.data(), sizeof(int) * ips, cudaMemcpyHostToDevice));
            f.items = items;
            CK(dalloc(plan, &f.head, (size_t)1));
            CK(dalloc(plan, &f.nact, (size_t)1));
            CK(dalloc(plan, &f.cnt, (size_t)3 * B));
            CK(dalloc(plan, &f.list, (size_t)B));
            CK(dalloc(plan, &f.ring, fused64_ring_elems(g)));
        } else {
            CK(dalloc(plan, &plan->W, (size_t)B * 3 * g.ax[2].P * g.NL));
        }
        if (g.split) CK(dalloc(plan, &g.Y, (size_t)B * 3 * g.ax[2].P * g.N1 * g.ax[1].P));
        CK(dalloc(plan, &plan->xbuf, (size_t)B * kd.vlen));
        CK(dalloc(plan, &plan->ybuf, (size_t)B * kd.vlen));
        CK(dalloc(plan, &ks.basis, (size_t)kd.ld * B * kd.vlen));
        CK(dalloc(plan, &ks.part, (size_t)B * kd.nchunk * 2 * kd.ld));
        CK(dalloc(plan, &ks.gram, (size_t)B * kd.ld * kd.ld));
        CK(dalloc(plan, &ks.hcol, (size_t)B * kd.ld));
        CK(dalloc(plan, &ks.R, (size_t)B * kd.ld * kd.mmax));
        CK(dalloc(plan, &ks.cs, (size_t)B * kd.mmax));
        CK(dalloc(plan, &ks.sn, (size_t)B * kd.mmax));
        CK(dalloc(plan, &ks.g, (size_t)B * kd.ld));
        CK(dalloc(plan, &ks.ycoef, (size_t)B * kd.mmax));
        CK(dalloc(plan, &ks.hist, (size_t)B * kd.mmax));
        CK(dalloc(plan, &ks.beta, (size_t)B));
        CK(dalloc(plan, &ks.bnorm, (size_t)B));
        CK(dalloc(plan, &ks.guess, (size_t)B));
        CK(dalloc(plan, &ks.rflag, (size_t)B));
        CK(dalloc(plan, &ks.running, (size_t)B));
        CK(dalloc(plan, &ks.fin, (size_t)B));
        CK(dalloc(plan, &ks.point, (size_t)B));
        CK(dalloc(plan, &ks.newv, (size_t)B));
        CK(dalloc(plan, &plan->d_refill_ctl, (size_t)2));
        CK(dalloc(plan, &plan->d_mesh_idx, (size_t)B));
        CK(dalloc(plan, &plan->d_mesh_nbr, (size_t)GSM_MESH_NNB * B));
        CK(dalloc(plan, &plan->d_mesh_wgt, (size_t)GSM_MESH_NNB * B));
        CK(dalloc(plan, &ks.scale, (size_t)B));
        CK(dalloc(plan, &ks.active, (size_t)B));
        CK(dalloc(plan, &ks.iters, (size_t)B));
        CK(dalloc(plan, &ks.nactive, (size_t)1));
        CK(dalloc(plan, &ks.pol, (size_t)B * 6));
        CK(dalloc(plan, &ks.tol, (size_t)1));
        CK(dalloc(plan, &plan->d_kvec, (size_t)B * 3));
        CK(dalloc(plan, &plan->d_k0, (size_t)B));
        CK(dalloc(plan, &plan->d_resid, (size_t)B));
        plan->pinned_bytes = sizeof(double) * ((size_t)B * (12 + kd.mmax) + 16);   // + 16: per-group read-back slots
        CK(cudaMallocHost(&plan->pinned, plan->pinned_bytes));
        CK(cudaEventCreateWithFlags(&plan->iter_ev[0], cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&plan->iter_ev[1], cudaEventDisableTiming));
        CK(dalloc(plan, &plan->d_gcount, (size_t)GSM_MAX_GROUPS));
        for (int q = 0; q < GSM_MAX_GROUPS; ++q) {
            if (q > 0) CK(cudaStreamCreateWithFlags(&plan->gstream[q], cudaStreamNonBlocking));
            CK(cudaEventCreateWithFlags(&plan->gev[q][0], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&plan->gev[q][1], cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&plan->gsync[q], cudaEventDisableTiming));
        }
        return GSM_OK;
    };
    st = body();
    if (st != GSM_OK) {
        g_create_error = plan->err;
        gsm_plan_destroy(plan);
        return st;
    }
    *out = plan;
    return GSM_OK;
}

extern "C" gsm_status gsm_plan_destroy(gsm_plan* plan) {
    if (!plan) return GSM_E_INVALID;
    cudaStreamSynchronize(plan->stream);
    plan->prof.destroy();
    for (cudaEvent_t e : plan->iter_ev) if (e) cudaEventDestroy(e);
    for (int q = 0; q < GSM_MAX_GROUPS; ++q) {
        if (plan->gstream[q]) { cudaStreamSynchronize(plan->gstream[q]); cudaStreamDestroy(plan->gstream[q]); }
        for (cudaEvent_t e : plan->gev[q]) if (e) cudaEventDestroy(e);
        if (plan->gsync[q]) cudaEventDestroy(plan->gsync[q]);
    }
    for (void* p : plan->allocs) cudaFree(p);
    if (plan->mesh_fields) cudaFree(plan->mesh_fields);
    if (plan->refill_buf) cudaFree(plan->refill_buf);
    if (plan->pinned) cudaFreeHost(plan->pinned);
    delete plan;
    return GSM_OK;
}

extern "C" gsm_status gsm_plan_coeffs(const gsm_plan* plan, double* host_out) {
    if (!plan || !host_out) return GSM_E_INVALID;
    const int* N = plan->desc.orders;
    const size_t ncoef = (size_t)(2 * N[0] - 1) * (2 * N[1] - 1) * (2 * N[2] - 1);
    CK(cudaStreamSynchronize(plan->stream));
    CK(cudaMemcpy(host_out, plan->coef, sizeof(cplx) * ncoef, cudaMemcpyDeviceToHost));
    return GSM_OK;
}

extern "C" gsm_status gsm_plan_info(const gsm_plan* plan, int fft_grid[3], long long* device_bytes, long long* launches) {
    if (!plan) return GSM_E_INVALID;
    if (fft_grid) for (int a = 0; a < 3; ++a) fft_grid[a] = plan->geom.ax[a].P;
    if (device_bytes) *device_bytes = plan->device_bytes;
    if (launches) {
        *launches = 0;
        for (int c = 0; c < KC_COUNT; ++c) *launches += plan->prof.launches[c];
    }
    return GSM_OK;
}

extern "C" const char* gsm_last_error(const gsm_plan* plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

// eps_b must keep k_m.k_m != k_b^2 for every kept m.  min over m of |k_m.k_m - k_b^2| / |k_b^2| on the
// host: k_m.k_m = a1(m1) + a2(m2) + a3(m3) is separable, so a sorted a3 and a binary search give O(N1 N2 log N3).
static bool singular_basis(const gsm_plan* plan, int batch, const double* kvec, const double* k0) {
    const ApplyGeom& g = plan->geom;
    const int N[3] = {g.N1, g.N2, g.N3};
    std::vector<double> a[3];
    for (int b = 0; b < batch; ++b) {
        const double kb2r = k0[b] * k0[b] * g.epsb_re, kb2i = k0[b] * k0[b] * g.epsb_im;
        const double mag = std::hypot(kb2r, kb2i);
        for (int ax = 0; ax < 3; ++ax) {
            a[ax].resize(N[ax]);
            for (int i = 0; i < N[ax]; ++i) {
                const double k = kvec[3 * b + ax] + (i + g.mmin[ax]) * g.K[ax];
                a[ax][i] = k * k;
            }
        }
        std::sort(a[2].begin(), a[2].end());
        double best = INFINITY;
        for (int i = 0; i < N[0]; ++i)
            for (int j = 0; j < N[1]; ++j) {
                const double target = kb2r - a[0][i] - a[1][j];
                auto it = std::lower_bound(a[2].begin(), a[2].end(), target);
                if (it != a[2].end()) best = std::min(best, std::fabs(*it - target));
                if (it != a[2].begin()) best = std::min(best, std::fabs(*(it - 1) - target));
            }
        const double dist = std::hypot(best, kb2i);
        if (!(dist > 1e-12 * mag) || !std::isfinite(dist)) return true;
    }
    return false;
}

extern "C" gsm_status gsm_apply(gsm_plan* plan, int batch, const double* k_bloch, const double* k0, const void* d_x,
                                void* d_y) {
    if (!plan) return GSM_E_INVALID;
    if (!k_bloch || !k0 || !d_x || !d_y || batch < 1 || batch > plan->max_batch || d_x == d_y)
        return fail(plan, GSM_E_INVALID, "gsm_apply: bad argument");
    if (singular_basis(plan, batch, k_bloch, k0)) return fail(plan, GSM_E_SINGULAR_BASIS, "k_m.k_m == k_b^2 for some m");
    CK(cudaMemcpyAsync(plan->d_kvec, k_bloch, sizeof(double) * 3 * batch, cudaMemcpyHostToDevice, plan->stream));
    CK(cudaMemcpyAsync(plan->d_k0, k0, sizeof(double) * batch, cudaMemcpyHostToDevice, plan->stream));
    CK(launch_apply(plan->geom, batch, plan->d_kvec, plan->d_k0, static_cast<const cplx*>(d_x), static_cast<cplx*>(d_y),
                    plan->W, &plan->fused, nullptr, plan->stream, &plan->prof, (double)batch));
    return GSM_OK;
}

// Plan-free, allocation-free operator apply (apply_static.cu); the failure text goes where gsm_last_error(NULL) finds it.
namespace gsm {
gsm_status apply_static(const double period[3], const int orders[3], double eps_b_re, double eps_b_im, int formulation,
                        const void* d_coef, int batch, const double* k_bloch, const double* k0, const void* d_x, void* d_y,
                        cudaStream_t st, std::string* err);
}
extern "C" gsm_status gsm_apply_static(const double period[3], const int orders[3], double eps_b_re, double eps_b_im,
                                       int formulation, const void* d_coef, int batch, const double* k_bloch,
                                       const double* k0, const void* d_x, void* d_y, void* cuda_stream) {
    std::string msg;
    const gsm_status st = gsm::apply_static(period, orders, eps_b_re, eps_b_im, formulation, d_coef, batch, k_bloch, k0, d_x,
                                            d_y, static_cast<cudaStream_t>(cuda_stream), &msg);
    return st < 0 ? fail(nullptr, st, msg.c_str()) : st;
}

// nb <= max_batch solves in lock step.  d_E: device [nb][vlen].  d_x0 (may be null, may alias d_E): initial guesses.
// Host outputs may be null.
static gsm_status run_batch(gsm_plan* plan, int nb, const double* kvec, const double* k0, const double* pol, double tol,
                            const cplx* d_x0, cplx* d_E, double* resp, int* iters, double* resid, double* hist,
                            int hist_cap, bool* not_converged) {
    const KrylovDims& kd = plan->kd;
    const KrylovState& ks = plan->ks;
    const ApplyGeom& g = plan->geom;
    cudaStream_t st = plan->stream;
    if (singular_basis(plan, nb, kvec, k0)) return fail(plan, GSM_E_SINGULAR_BASIS, "k_m.k_m == k_b^2 for some m");
    plan->last_nb = nb;
    double* pin = static_cast<double*>(plan->pinned);
    CK(cudaMemcpyAsync(plan->d_kvec, kvec, sizeof(double) * 3 * nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(plan->d_k0, k0, sizeof(double) * nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ks.pol, pol, sizeof(double) * 6 * nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ks.tol, &tol, sizeof(double), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ks.nactive, &nb, sizeof(int), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(ks.basis, 0, sizeof(cplx) * (size_t)nb * kd.vlen, st));
    Profiler* prof = &plan->prof;
    CK(launch_krylov_init(kd, ks, nb, plan->i0, g.n, st, prof));
    const size_t vs = (size_t)nb * kd.vlen;
    if (d_x0) {   // r0 = b - A x0 (one more apply), v_0 = r0 / ||r0||; GMRES then solves A d = r0 and E = x0 + d
        CK(launch_apply(g, nb, plan->d_kvec, plan->d_k0, d_x0, ks.basis + vs, plan->W, &plan->fused, nullptr, st, prof,
                        (double)nb));
        CK(launch_krylov_guess(kd, ks, nb, plan->i0, g.n, st, prof));
    }
    // Launches of the iteration loop are billed (algorithmic bytes) after the batch, from the final iteration counts:
    // the host learns how many solves were still iterating one iteration late.
    //
    // Groups.  The Arnoldi kernel is HBM-bound and its clusters occupy 112 of the 148 SMs; the plane convolution of the
    // apply is bound by the fp64 and shared-memory pipes and leaves HBM idle; and small batches leave every kernel
    // latency-bound.  The batch is therefore cut into up to GSM_MAX_GROUPS groups of consecutive solves that iterate on
    // streams of their own, so that one group's Gram-Schmidt runs beside another group's apply (the groups drift apart
    // by themselves; forcing a stagger, or a high-priority stream for the Gram-Schmidt launches, changes nothing).
    // Per solve nothing changes (same kernels, same reductions: bit-identical results).  One group when per-launch
    // profiling is on (clean kernel times), on the two-sweep and fused-apply paths, and below 8 solves.
    int G = 1;   // measured at 31^3 (ms per scan, 1 / 2 / 4 groups): 16 solves 11.1 / 9.7 / 9.1, 64: 35.4 / 32.2 / 32.9, 256: 129 / 125 / 127
    if (plan->mgs_cs > 0 && !plan->fused.ring && !prof->on && nb >= 8) G = nb >= 48 ? 2 : std::min(GSM_MAX_GROUPS, nb / 4);
    GroupBounds gb{};
    for (int q = 0; q <= G; ++q) gb.b[q] = (int)((long)nb * q / G);
    KrylovDims kdg = kd;
    kdg.vstride = (long)vs;
    int* gpin = reinterpret_cast<int*>(pin + (size_t)plan->max_batch * (12 + kd.mmax));   // [group][parity]
    if (G > 1) {
        CK(launch_group_count(ks, G, gb, plan->d_gcount, st, prof));
        CK(cudaEventRecord(plan->gsync[0], st));
        for (int q = 1; q < G; ++q) CK(cudaStreamWaitEvent(plan->gstream[q], plan->gsync[0], 0));
    }
    bool done[GSM_MAX_GROUPS] = {};
    for (int j = 0; j < kd.mmax; ++j) {
        for (int q = 0; q < G; ++q) {
            if (done[q]) continue;
            const int b0 = gb.b[q], gn = gb.b[q + 1] - b0;
            cudaStream_t sq = q == 0 ? st : plan->gstream[q];
            const KrylovState kq = G > 1 ? krylov_state_view(kd, ks, b0, plan->d_gcount + q) : ks;
            ApplyGeom gq = g;
            if (gq.Y) gq.Y += (size_t)b0 * 3 * g.ax[2].P * g.N1 * g.ax[1].P;
            cplx* Wq = plan->W ? plan->W + (size_t)b0 * 3 * g.ax[2].P * g.NL : nullptr;
            const cplx* xq = ks.basis + (size_t)j * vs + (size_t)b0 * kd.vlen;
            CK(launch_apply(gq, gn, plan->d_kvec + 3 * b0, plan->d_k0 + b0, xq, const_cast<cplx*>(xq) + vs, Wq, &plan->fused,
                            kq.active, sq, prof, 0.0));
            if (plan->mgs_cs > 0) {
                CK(launch_arnoldi_cluster(kdg, kq, gn, j, plan->mgs_cs, plan->mgs_chunk, plan->mgs_nclusters, sq, prof));
            } else {
                CK(launch_sweep_dots(kd, ks, nb, j, st, prof));
                CK(launch_hsolve(kd, ks, nb, j, st, prof));
                CK(launch_sweep_update(kd, ks, nb, j, st, prof));
                CK(launch_givens(kd, ks, nb, j, st, prof));
                CK(launch_normalize(kd, ks, nb, j, st, prof));
            }
            // The count of solves still iterating comes back one iteration late: iteration j + 1 is enqueued before the
            // host looks at the count after iteration j - 1, so launches never wait for a round trip.  If everything had
            // already converged, the extra iteration's CTAs find their `active` flags cleared and exit at once.
            CK(cudaMemcpyAsync(gpin + 2 * q + (j & 1), kq.nactive, sizeof(int), cudaMemcpyDeviceToHost, sq));
            CK(cudaEventRecord(plan->gev[q][j & 1], sq));
        }
        bool all = true;
        for (int q = 0; q < G; ++q) {
            if (!done[q] && j >= 1) {
                CK(cudaEventSynchronize(plan->gev[q][(j - 1) & 1]));
                if (gpin[2 * q + ((j - 1) & 1)] <= 0) done[q] = true;
            }
            all = all && done[q];
        }
        if (all) break;
    }
    for (int q = 1; q < G; ++q) {   // join
        CK(cudaEventRecord(plan->gsync[q], plan->gstream[q]));
        CK(cudaStreamWaitEvent(st, plan->gsync[q], 0));
    }
    CK(launch_backsolve(kd, ks, nb, st, prof));
    CK(launch_combine(kd, ks, nb, d_x0, d_E, st, prof));
    // true residual with one more apply; a guess that was accepted without iterating has it already
    CK(launch_residual_select(kd, ks, nb, st, prof));
    CK(launch_apply(g, nb, plan->d_kvec, plan->d_k0, d_E, plan->ybuf, plan->W, &plan->fused, ks.rflag, st, prof, 0.0));
    CK(launch_true_residual(kd, ks, nb, plan->ybuf, plan->i0, g.n, plan->d_resid, st, prof));
    int* h_iters = reinterpret_cast<int*>(pin + 2);
    double* h_resid = pin + 2 + nb;           // ints occupy at most nb doubles
    int* h_active = reinterpret_cast<int*>(pin + 2 + 2 * (size_t)nb);
    double* h_resp = pin + 2 + 3 * (size_t)nb;
    CK(cudaMemcpyAsync(h_iters, ks.iters, sizeof(int) * nb, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_resid, plan->d_resid, sizeof(double) * nb, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_active, ks.active, sizeof(int) * nb, cudaMemcpyDeviceToHost, st));
    int* h_rflag = reinterpret_cast<int*>(pin + 2 + 9 * (size_t)nb + kd.mmax);
    CK(cudaMemcpyAsync(h_rflag, ks.rflag, sizeof(int) * nb, cudaMemcpyDeviceToHost, st));
    // E at m = 0: three complex numbers per solve, stride n inside a vector
    CK(cudaMemcpy2DAsync(h_resp, sizeof(cplx), d_E + plan->i0, sizeof(cplx) * g.n, sizeof(cplx), (size_t)3 * nb,
                         cudaMemcpyDeviceToHost, st));
    if (hist && hist_cap > 0)
        CK(cudaMemcpyAsync(pin + 2 + 9 * (size_t)nb, ks.hist, sizeof(double) * std::min(hist_cap, kd.mmax),
                           cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    {   // bill the iteration loop: solve b ran iterations j = 0 .. m_b - 1, each one apply and one Arnoldi step
        double s1 = 0.0, s2 = 0.0, nres = 0.0;   // sum m_b, sum m_b (m_b - 1) / 2, applies of the residual check
        for (int b = 0; b < nb; ++b) { const double m = h_iters[b]; s1 += m; s2 += 0.5 * m * (m - 1.0); nres += h_rflag[b]; }
        const double V = 16.0 * kd.vlen;
        bill_apply(g, plan->fused.ring != nullptr, prof, s1 + nres);
        if (plan->mgs_cs > 0) {
            prof->bytes[KC_ARNOLDI_MGS] += V * (s2 + 3.0 * s1);       // (j + 3) V: w, v_0..v_j, write v_{j+1}
        } else {
            prof->bytes[KC_SWEEP_DOTS] += V * (s2 + 2.0 * s1);        // (j + 2) V
            prof->bytes[KC_SWEEP_UPDATE] += V * (s2 + 3.0 * s1);      // (j + 3) V
            prof->bytes[KC_NORMALIZE] += V * 2.0 * s1;
        }
        prof->bytes[KC_COMBINE] += V * (s1 + nb);                     // x = sum y_i v_i: m_b reads, one write
    }
    for (int b = 0; b < nb; ++b) {
        if (iters) iters[b] = h_iters[b];
        if (resid) resid[b] = h_resid[b];
        if (h_active[b]) *not_converged = true;
        if (resp) for (int q = 0; q < 6; ++q) resp[6 * b + q] = h_resp[6 * b + q];
    }
    if (hist && hist_cap > 0) {
        const int cnt = std::min(std::min(hist_cap, kd.mmax), h_iters[0]);
        for (int q = 0; q < cnt; ++q) hist[q] = pin[2 + 9 * (size_t)nb + q];
    }
    return GSM_OK;
}

// Slot-refill scan from a zero start (npts > max_batch, cluster Gram-Schmidt path): max_batch slots run in lock step, each
// at its own Arnoldi index; a slot whose solve has finished (true residual checked with one more apply, results recorded
// under its point index) takes the next pending point at the next tick.  Per solve the arithmetic is that of run_batch.
static gsm_status run_refill(gsm_plan* plan, int npts, const double* kvec, const double* k0, const double* pol, double tol,
                             cplx* d_E_out, double* resp, int* iters, double* resid, bool* not_converged) {
    const KrylovDims& kd = plan->kd;
    const KrylovState& ks = plan->ks;
    cudaStream_t st = plan->stream;
    Profiler* prof = &plan->prof;
    const int B = plan->max_batch;
    if (singular_basis(plan, npts, kvec, k0)) return fail(plan, GSM_E_SINGULAR_BASIS, "k_m.k_m == k_b^2 for some m");
    plan->last_nb = 0;   // slots are reused: no per-solve history is kept
    // device copy of the list and per-point outputs: [resp 6][kvec 3][k0 1][pol 6][resid 1] doubles, [iters][flag] ints
    const size_t per_pt = sizeof(double) * 17 + sizeof(int) * 2;
    if (plan->refill_cap < (size_t)npts) {
        if (plan->refill_buf) cudaFree(plan->refill_buf);
        plan->device_bytes -= (long long)(per_pt * plan->refill_cap);
        plan->refill_buf = nullptr;
        plan->refill_cap = 0;
        CK(cudaMalloc(&plan->refill_buf, per_pt * (size_t)npts));
        plan->refill_cap = (size_t)npts;
        plan->device_bytes += (long long)(per_pt * plan->refill_cap);
    }
    double* dd = static_cast<double*>(plan->refill_buf);
    cplx* d_resp = reinterpret_cast<cplx*>(dd);   // first: 16-byte aligned for any npts
    double *d_kv = dd + 6 * (size_t)npts, *d_k0 = dd + 9 * (size_t)npts, *d_pol = dd + 10 * (size_t)npts, *d_res = dd + 16 * (size_t)npts;
    int* d_it = reinterpret_cast<int*>(dd + 17 * (size_t)npts);
    int* d_flag = d_it + npts;
    CK(cudaMemcpyAsync(d_kv, kvec, sizeof(double) * 3 * npts, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_k0, k0, sizeof(double) * npts, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_pol, pol, sizeof(double) * 6 * npts, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ks.tol, &tol, sizeof(double), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(ks.nactive, 0, sizeof(int), st));
    CK(cudaMemsetAsync(plan->d_refill_ctl, 0, 2 * sizeof(int), st));
    for (int* flags : {ks.running, ks.fin, ks.active, ks.newv, ks.rflag}) CK(cudaMemsetAsync(flags, 0, sizeof(int) * B, st));
    RefillDev r{d_kv, d_k0, d_pol, npts, plan->d_refill_ctl, plan->d_refill_ctl + 1, d_it, d_res, d_resp, d_flag};
    ApplyGeom gs = plan->geom;            // the Arnoldi applies: x = v_{j_b}, y = slot j_b + 1 of the basis pool
    gs.jslot = ks.iters;
    gs.jstride = (long)B * kd.vlen;
    const size_t vs = (size_t)B * kd.vlen;
    int* pin_i = static_cast<int*>(plan->pinned);
    // first fill: every slot is free
    CK(launch_refill_commit(kd, ks, r, B, plan->i0, plan->geom.n, plan->xbuf, plan->d_resid, plan->d_kvec, plan->d_k0, st, prof));
    const long max_ticks = ((long)npts / B + 2) * ((long)kd.mmax + 2);
    for (long t = 0; t < max_ticks; ++t) {
        CK(launch_apply(gs, B, plan->d_kvec, plan->d_k0, ks.basis, ks.basis + vs, plan->W, &plan->fused, ks.active, st, prof, 0.0));
        CK(launch_arnoldi_cluster(kd, ks, B, -1, plan->mgs_cs, plan->mgs_chunk, plan->mgs_nclusters, st, prof));
        // solves that finished in this tick: x = sum y_i v_i, true residual with one more apply, results recorded, slot refilled
        CK(launch_refill_mark(kd, ks, B, st, prof));
        CK(launch_backsolve(kd, ks, B, st, prof, ks.fin));
        CK(launch_combine(kd, ks, B, nullptr, plan->xbuf, st, prof, ks.fin));
        CK(launch_apply(plan->geom, B, plan->d_kvec, plan->d_k0, plan->xbuf, plan->ybuf, plan->W, &plan->fused, ks.rflag, st, prof, 0.0));
        CK(launch_true_residual(kd, ks, B, plan->ybuf, plan->i0, plan->geom.n, plan->d_resid, st, prof));
        if (d_E_out) CK(launch_mesh_scatter(kd, B, plan->xbuf, ks.point, d_E_out, st, prof, ks.fin));
        CK(launch_refill_commit(kd, ks, r, B, plan->i0, plan->geom.n, plan->xbuf, plan->d_resid, plan->d_kvec, plan->d_k0, st, prof));
        // the count of recorded points comes back one tick late, so that no launch waits for a round trip
        CK(cudaMemcpyAsync(pin_i + (t & 1), r.ndone, sizeof(int), cudaMemcpyDeviceToHost, st));
        CK(cudaEventRecord(plan->iter_ev[t & 1], st));
        if (t >= 1) {
            CK(cudaEventSynchronize(plan->iter_ev[(t - 1) & 1]));
            if (pin_i[(t - 1) & 1] >= npts) break;
        }
    }
    std::vector<int> h_it(npts), h_flag(npts);
    std::vector<double> h_res(npts), h_resp(6 * (size_t)npts);
    CK(cudaMemcpyAsync(h_it.data(), d_it, sizeof(int) * npts, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_flag.data(), d_flag, sizeof(int) * npts, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_res.data(), d_res, sizeof(double) * npts, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_resp.data(), d_resp, sizeof(cplx) * 3 * npts, cudaMemcpyDeviceToHost, st));
    int done = 0;
    CK(cudaMemcpyAsync(&done, r.ndone, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (done < npts) return fail(plan, GSM_E_CUDA, "slot-refill scan ended before every point was solved");
    double s1 = 0.0, s2 = 0.0;
    for (int p = 0; p < npts; ++p) {
        const double m = h_it[p];
        s1 += m;
        s2 += 0.5 * m * (m - 1.0);
        if (iters) iters[p] = h_it[p];
        if (resid) resid[p] = h_res[p];
        if (h_flag[p]) *not_converged = true;
        if (resp) for (int q = 0; q < 6; ++q) resp[6 * (size_t)p + q] = h_resp[6 * (size_t)p + q];
    }
    const double V = 16.0 * kd.vlen;
    bill_apply(plan->geom, false, prof, s1 + npts);
    prof->bytes[KC_ARNOLDI_MGS] += V * (s2 + 3.0 * s1);
    prof->bytes[KC_COMBINE] += V * (s1 + npts);
    return GSM_OK;
}

extern "C" gsm_status gsm_solve(gsm_plan* plan, const double k_bloch[3], double k0, const double pol[6], double tol,
                                void* d_E_out, double* resid_hist_host, int hist_cap, int* n_iters,
                                double* true_rel_resid) {
    if (!plan) return GSM_E_INVALID;
    if (!k_bloch || !pol || !d_E_out || !(tol > 0.0)) return fail(plan, GSM_E_INVALID, "gsm_solve: bad argument");
    bool nc = false;
    gsm_status s = run_batch(plan, 1, k_bloch, &k0, pol, tol, nullptr, static_cast<cplx*>(d_E_out), nullptr, n_iters,
                             true_rel_resid, resid_hist_host, hist_cap, &nc);
    if (s != GSM_OK) return s;
    return nc ? GSM_NOT_CONVERGED : GSM_OK;
}

extern "C" gsm_status gsm_plan_history(gsm_plan* plan, int b, double* resid_hist_host, int hist_cap, int* n_iters) {
    if (!plan) return GSM_E_INVALID;
    if (b < 0 || b >= plan->last_nb || hist_cap < 0 || (hist_cap > 0 && !resid_hist_host) || !n_iters)
        return fail(plan, GSM_E_INVALID, "gsm_plan_history: bad argument or no such solve in the last batch");
    CK(cudaStreamSynchronize(plan->stream));
    int m = 0;
    CK(cudaMemcpy(&m, plan->ks.iters + b, sizeof(int), cudaMemcpyDeviceToHost));
    const int cnt = std::min(std::min(hist_cap, plan->kd.mmax), m);
    if (cnt > 0)
        CK(cudaMemcpy(resid_hist_host, plan->ks.hist + (size_t)b * plan->kd.mmax, sizeof(double) * cnt, cudaMemcpyDeviceToHost));
    *n_iters = m;
    return GSM_OK;
}

extern "C" gsm_status gsm_scan_guess(gsm_plan* plan, int npts, const double* k_bloch, const double* k0, const double* pol,
                                     double tol, const void* d_x0, double* resp_host, int* iters, double* resid,
                                     void* d_E_out) {
    if (!plan) return GSM_E_INVALID;
    if (npts < 0 || !k_bloch || !k0 || !pol || !(tol > 0.0)) return fail(plan, GSM_E_INVALID, "gsm_scan: bad argument");
    bool nc = false;
    if ((plan->desc.flags & GSM_FLAG_SLOT_REFILL) && !d_x0 && npts > plan->max_batch && plan->mgs_cs > 0 && !plan->fused.ring) {
        gsm_status s = run_refill(plan, npts, k_bloch, k0, pol, tol, static_cast<cplx*>(d_E_out), resp_host, iters, resid, &nc);
        if (s != GSM_OK) return s;
        return nc ? GSM_NOT_CONVERGED : GSM_OK;
    }
    for (int p0 = 0; p0 < npts; p0 += plan->max_batch) {
        const int nb = std::min(plan->max_batch, npts - p0);
        cplx* dE = d_E_out ? static_cast<cplx*>(d_E_out) + (size_t)p0 * plan->kd.vlen : plan->xbuf;
        const cplx* x0 = d_x0 ? static_cast<const cplx*>(d_x0) + (size_t)p0 * plan->kd.vlen : nullptr;
        gsm_status s = run_batch(plan, nb, k_bloch + 3 * (size_t)p0, k0 + p0, pol + 6 * (size_t)p0, tol, x0, dE,
                                 resp_host ? resp_host + 6 * (size_t)p0 : nullptr, iters ? iters + p0 : nullptr,
                                 resid ? resid + p0 : nullptr, nullptr, 0, &nc);
        if (s != GSM_OK) return s;
    }
    return nc ? GSM_NOT_CONVERGED : GSM_OK;
}

extern "C" gsm_status gsm_scan(gsm_plan* plan, int npts, const double* k_bloch, const double* k0, const double* pol,
                               double tol, double* resp_host, int* iters, double* resid, void* d_E_out) {
    return gsm_scan_guess(plan, npts, k_bloch, k0, pol, tol, nullptr, resp_host, iters, resid, d_E_out);
}

// Lagrange weights at position t of the interpolation nodes tn[0..cnt)
static void lagrange_weights(double t, const int* tn, int cnt, double* w) {
    for (int a = 0; a < cnt; ++a) {
        double v = 1.0;
        for (int b = 0; b < cnt; ++b)
            if (b != a) v *= (t - tn[b]) / (double)(tn[a] - tn[b]);
        w[a] = v;
    }
}

// Wave structure of gsm_scan_mesh (reading R25).  levels is first reduced so that wave 0 holds at least two points.
static int mesh_levels(int npts, int levels) {
    while (levels > 1 && (1 << (levels - 1)) >= npts) --levels;
    return levels;
}
// Interpolation stencil of point p when the multiples of S are solved: the nearest GSM_MESH_NNB of them (towards an end
// of the list the missing side is made up from the other one) and their Lagrange weights at p.
static int mesh_stencil(int p, int S, int npts, int* nodes, double* w) {
    const int last = ((npts - 1) / S) * S;
    int lo = (p / S) * S, hi = lo + S, cnt = 0;
    while (cnt < GSM_MESH_NNB && (lo >= 0 || hi <= last)) {
        const bool take_lo = lo >= 0 && (hi > last || p - lo <= hi - p);
        if (take_lo) { nodes[cnt++] = lo; lo -= S; } else { nodes[cnt++] = hi; hi += S; }
    }
    lagrange_weights((double)p, nodes, cnt, w);
    return cnt;
}
// Points of the next wave when the multiples of S are solved: the odd multiples of S / 2, or - `collapse` - every point
// that is not solved yet.  Returns the stride of the solved set afterwards.
static int mesh_wave(int npts, int S, bool collapse, std::vector<int>& targets) {
    targets.clear();
    if (collapse) {
        for (int p = 0; p < npts; ++p)
            if (p % S) targets.push_back(p);
        return 1;
    }
    for (int p = S / 2; p < npts; p += S) targets.push_back(p);
    return S / 2;
}

extern "C" gsm_status gsm_mesh_schedule(int npts, int levels, int collapse_after, int* wave, int* nodes, double* weights) {
    if (npts < 0 || levels < 1 || levels > 16 || !wave || !nodes || !weights) return GSM_E_INVALID;
    if (npts == 0) return GSM_OK;
    levels = mesh_levels(npts, levels);
    int S = 1 << (levels - 1);
    for (int p = 0; p < npts; ++p) {
        wave[p] = p % S ? -1 : 0;
        for (int q = 0; q < GSM_MESH_NNB; ++q) { nodes[(size_t)GSM_MESH_NNB * p + q] = -1; weights[(size_t)GSM_MESH_NNB * p + q] = 0.0; }
    }
    std::vector<int> targets;
    for (int w = 1; S > 1; ++w) {
        const int Sn = S;
        S = mesh_wave(npts, Sn, collapse_after > 0 && w > collapse_after, targets);
        for (int p : targets) {
            wave[p] = w;
            int nd[GSM_MESH_NNB];
            double wt[GSM_MESH_NNB];
            const int cnt = mesh_stencil(p, Sn, npts, nd, wt);
            for (int q = 0; q < cnt; ++q) { nodes[(size_t)GSM_MESH_NNB * p + q] = nd[q]; weights[(size_t)GSM_MESH_NNB * p + q] = wt[q]; }
        }
    }
    return GSM_OK;
}

extern "C" gsm_status gsm_scan_mesh(gsm_plan* plan, int npts, const double* k_bloch, const double* k0, const double* pol,
                                    double tol, int levels, double* resp_host, int* iters, double* resid, void* d_E_out) {
    if (!plan) return GSM_E_INVALID;
    if (npts < 0 || !k_bloch || !k0 || !pol || !(tol > 0.0) || levels < 1 || levels > 16)
        return fail(plan, GSM_E_INVALID, "gsm_scan_mesh: bad argument");
    if (npts == 0) return GSM_OK;
    levels = mesh_levels(npts, levels);
    const size_t vlen = (size_t)plan->kd.vlen;
    cplx* all = static_cast<cplx*>(d_E_out);
    if (!all) {
        if (plan->mesh_cap < (size_t)npts) {
            if (plan->mesh_fields) cudaFree(plan->mesh_fields);
            plan->device_bytes -= (long long)(sizeof(cplx) * vlen * plan->mesh_cap);
            plan->mesh_fields = nullptr;
            plan->mesh_cap = 0;
            CK(cudaMalloc(reinterpret_cast<void**>(&plan->mesh_fields), sizeof(cplx) * vlen * npts));
            plan->mesh_cap = (size_t)npts;
            plan->device_bytes += (long long)(sizeof(cplx) * vlen * plan->mesh_cap);
        }
        all = plan->mesh_fields;
    }
    const int B = plan->max_batch;
    const int NNB = GSM_MESH_NNB;
    std::vector<double> kb(3 * (size_t)B), kk(B), pl(6 * (size_t)B), wgt(2 * (size_t)NNB * B), h_resp(6 * (size_t)B), h_resid(B);
    std::vector<int> idx(B), nbr((size_t)NNB * B), h_iters(B), targets;
    std::vector<double> xi_all(2 * (size_t)npts, 0.0);   // response projected on the amplitude, for the pole estimate
    bool nc = false;
    int S = 1 << (levels - 1);        // the multiples of S are solved (after wave 0)
    for (int p = 0; p < npts; p += S) targets.push_back(p);
    double prev_mean = -1.0;          // mean iteration count of the previous guessed wave
    for (int w = 0; w == 0 || S > 1; ++w) {
        // Wave 0: the multiples of S from x0 = 0.  Wave w: the points mid-way between the solved ones, guessed from
        // the nearest solved points - or, once a guessed wave has needed no more than one iteration per point on
        // average (the guesses are already at the solver tolerance), every remaining point at once.
        const int Sn = S;             // stride of the solved set the stencils draw from
        if (w > 0) S = mesh_wave(npts, Sn, prev_mean >= 0.0 && prev_mean <= 1.0, targets);
        // Near a pole eta of the response the field behaves as R / (kappa - eta) + smooth, which
        // polynomial interpolation follows badly - and those are the points that need most iterations.  The solved
        // points (multiples of Sn: an equidistant mesh) give the poles in units of the list index through the pole
        // search of Eq. 7-10; the guess then interpolates prod_k (t - eta_k) E(t), which is smooth, and divides the
        // product out at the target.  Only the guess changes: the solves and their stop test do not.
        const int Np = 5, Nd = 10;
        double pe[2 * Np];
        int npole = 0;
        const int cnt0 = w > 0 ? (npts - 1) / Sn + 1 : 0;     // solved points so far
        if (w > 0 && cnt0 >= Np + Nd) {
            std::vector<double> tt(cnt0), xs(2 * (size_t)cnt0);
            for (int i = 0; i < cnt0; ++i) {
                tt[i] = (double)Sn * i;
                xs[2 * i] = xi_all[2 * (size_t)Sn * i];
                xs[2 * i + 1] = xi_all[2 * (size_t)Sn * i + 1];
            }
            double eta[2 * Np], zeta[2 * Np];
            int best = -1;
            if (gsm_pole_search(cnt0, tt.data(), xs.data(), Np, Nd, tt.front(), tt.back(), eta, zeta, &best) == GSM_OK && best >= 0) {
                const double zmax = std::hypot(zeta[2 * best], zeta[2 * best + 1]);
                for (int k = 0; k < Np; ++k)      // every pole inside the mesh whose amplitude matters
                    if (eta[2 * k] >= tt.front() && eta[2 * k] <= tt.back() &&
                        std::hypot(zeta[2 * k], zeta[2 * k + 1]) >= 1e-6 * zmax) {
                        pe[2 * npole] = eta[2 * k];
                        pe[2 * npole + 1] = eta[2 * k + 1];
                        ++npole;
                    }
            }
        }
        double wave_iters = 0.0;
        for (size_t t0 = 0; t0 < targets.size(); t0 += (size_t)B) {
            const int nb = (int)std::min((size_t)B, targets.size() - t0);
            for (int b = 0; b < nb; ++b) {
                const int p = targets[t0 + b];
                idx[b] = p;
                for (int a = 0; a < 3; ++a) kb[3 * b + a] = k_bloch[3 * (size_t)p + a];
                kk[b] = k0[p];
                for (int q = 0; q < 6; ++q) pl[6 * b + q] = pol[6 * (size_t)p + q];
                if (w > 0) {
                    int nodes[GSM_MESH_NNB];
                    double wl[GSM_MESH_NNB];
                    const int cnt = mesh_stencil(p, Sn, npts, nodes, wl);
                    for (int q = 0; q < NNB; ++q) {
                        nbr[NNB * b + q] = q < cnt ? nodes[q] : -1;
                        double wr = q < cnt ? wl[q] : 0.0, wi = 0.0;
                        for (int k = 0; k < npole && q < cnt; ++k) {   // times (t_q - eta_k) / (t_p - eta_k)
                            const double ar = nodes[q] - pe[2 * k], ai = -pe[2 * k + 1];
                            const double br = p - pe[2 * k], bi = -pe[2 * k + 1];
                            const double inv = 1.0 / (br * br + bi * bi);
                            const double fr = (ar * br + ai * bi) * inv, fi = (ai * br - ar * bi) * inv;
                            const double tr = wr * fr - wi * fi;
                            wi = wr * fi + wi * fr;
                            wr = tr;
                        }
                        if (!std::isfinite(wr) || !std::isfinite(wi)) { wr = q < cnt ? wl[q] : 0.0; wi = 0.0; }
                        wgt[2 * (NNB * b + q)] = wr;
                        wgt[2 * (NNB * b + q) + 1] = wi;
                    }
                }
            }
            cudaStream_t st = plan->stream;
            CK(cudaMemcpyAsync(plan->d_mesh_idx, idx.data(), sizeof(int) * nb, cudaMemcpyHostToDevice, st));
            const cplx* x0 = nullptr;
            if (w > 0) {
                CK(cudaMemcpyAsync(plan->d_mesh_nbr, nbr.data(), sizeof(int) * NNB * nb, cudaMemcpyHostToDevice, st));
                CK(cudaMemcpyAsync(plan->d_mesh_wgt, wgt.data(), sizeof(cplx) * NNB * nb, cudaMemcpyHostToDevice, st));
                CK(launch_mesh_guess(plan->kd, nb, all, plan->d_mesh_nbr, plan->d_mesh_wgt, plan->xbuf, st, &plan->prof));
                CK(cudaStreamSynchronize(st));   // the host vectors are rewritten by the next chunk
                x0 = plan->xbuf;
            }
            gsm_status s2 = run_batch(plan, nb, kb.data(), kk.data(), pl.data(), tol, x0, plan->xbuf, h_resp.data(),
                                      h_iters.data(), h_resid.data(), nullptr, 0, &nc);
            if (s2 != GSM_OK) return s2;
            CK(launch_mesh_scatter(plan->kd, nb, plan->xbuf, plan->d_mesh_idx, all, st, &plan->prof));
            CK(cudaStreamSynchronize(st));
            for (int b = 0; b < nb; ++b) {
                const size_t p = (size_t)idx[b];
                if (resp_host) for (int q = 0; q < 6; ++q) resp_host[6 * p + q] = h_resp[6 * b + q];
                {   // xi = sum_c conj(a_c) E_c / |a|^2
                    const double* a = pol + 6 * p;
                    double re = 0.0, im = 0.0, nrm = 0.0;
                    for (int c = 0; c < 3; ++c) {
                        re += a[2 * c] * h_resp[6 * b + 2 * c] + a[2 * c + 1] * h_resp[6 * b + 2 * c + 1];
                        im += a[2 * c] * h_resp[6 * b + 2 * c + 1] - a[2 * c + 1] * h_resp[6 * b + 2 * c];
                        nrm += a[2 * c] * a[2 * c] + a[2 * c + 1] * a[2 * c + 1];
                    }
                    xi_all[2 * p] = nrm > 0.0 ? re / nrm : 0.0;
                    xi_all[2 * p + 1] = nrm > 0.0 ? im / nrm : 0.0;
                }
                wave_iters += h_iters[b];
                if (iters) iters[p] = h_iters[b];
                if (resid) resid[p] = h_resid[b];
            }
        }
        if (w > 0 && !targets.empty()) prev_mean = wave_iters / (double)targets.size();
    }
    return nc ? GSM_NOT_CONVERGED : GSM_OK;
}


// ---- profiler (gsm_plan_profile / gsm_plan_profile_read) ---------------------------------------------------------
namespace gsm {
static const char* const kKernelClassNames[KC_COUNT] = {
    "z_forward", "xy_conv", "z_inverse_green", "sweep_dots", "hsolve", "sweep_update", "givens", "normalize",
    "arnoldi_mgs", "combine", "residual", "small", "plan", "apply_fused"};
const char* kernel_class_name(int cls) { return cls >= 0 && cls < KC_COUNT ? kKernelClassNames[cls] : ""; }

void Profiler::begin(int c, cudaStream_t st, double nbytes) {
    launches[c] += 1;
    bytes[c] += nbytes;
    if (!on) return;
    if (2 * used + 1 >= ev.size()) {
        cudaEvent_t a = nullptr, b = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { on = false; return; }
        ev.push_back(a);
        ev.push_back(b);
        cls.push_back(c);
    }
    cls[used] = c;
    cudaEventRecord(ev[2 * used], st);
}
void Profiler::end(cudaStream_t st) {
    if (!on) return;
    cudaEventRecord(ev[2 * used + 1], st);
    ++used;
}
cudaError_t Profiler::collect() {
    for (size_t i = 0; i < used; ++i) {
        cudaError_t e = cudaEventSynchronize(ev[2 * i + 1]);
        if (e != cudaSuccess) return e;
        float t = 0.f;
        e = cudaEventElapsedTime(&t, ev[2 * i], ev[2 * i + 1]);
        if (e != cudaSuccess) return e;
        ms[cls[i]] += (double)t;
    }
    used = 0;
    return cudaSuccess;
}
void Profiler::reset() {
    used = 0;
    for (int c = 0; c < KC_COUNT; ++c) { launches[c] = 0; ms[c] = 0.0; bytes[c] = 0.0; }
}
void Profiler::destroy() {
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    ev.clear();
    cls.clear();
    used = 0;
}
}  // namespace gsm

extern "C" gsm_status gsm_plan_profile(gsm_plan* plan, int enable) {
    if (!plan) return GSM_E_INVALID;
    CK(cudaStreamSynchronize(plan->stream));
    CK(plan->prof.collect());
    plan->prof.on = enable != 0;
    return GSM_OK;
}

extern "C" int gsm_kernel_class_count(void) { return KC_COUNT; }
extern "C" const char* gsm_kernel_class_name(int cls) { return kernel_class_name(cls); }

extern "C" gsm_status gsm_plan_profile_read(gsm_plan* plan, int ncls, long long* launches, double* ms, double* bytes,
                                            int reset) {
    if (!plan || ncls < 0) return GSM_E_INVALID;
    CK(cudaStreamSynchronize(plan->stream));
    CK(plan->prof.collect());
    for (int c = 0; c < ncls && c < KC_COUNT; ++c) {
        if (launches) launches[c] = plan->prof.launches[c];
        if (ms) ms[c] = plan->prof.ms[c];
        if (bytes) bytes[c] = plan->prof.bytes[c];
    }
    if (reset) plan->prof.reset();
    return GSM_OK;
}

// Replace the cell (shapes or voxel grid, permittivities, periods) of an existing plan without reallocating the
// workspaces: re-runs step a0 (coefficients and their spectrum).  orders must be unchanged.
extern "C" gsm_status gsm_plan_set_cell(gsm_plan* plan, const gsm_plan_desc* desc) {
    if (!plan) return GSM_E_INVALID;
    if (!desc) return fail(plan, GSM_E_INVALID, "gsm_plan_set_cell: null descriptor");
    for (int a = 0; a < 3; ++a) {
        if (desc->orders[a] != plan->desc.orders[a]) return fail(plan, GSM_E_INVALID, "gsm_plan_set_cell: orders differ");
        if (!(desc->period[a] > 0.0)) return fail(plan, GSM_E_INVALID, "periods must be positive");
    }
    if (desc->eps_b_re == 0.0 && desc->eps_b_im == 0.0) return fail(plan, GSM_E_INVALID, "eps_b must be non-zero");
    if (desc->eps_grid_host == nullptr && (desc->n_shapes < 0 || (desc->n_shapes > 0 && !desc->shapes)))
        return fail(plan, GSM_E_INVALID, "shapes missing");
    if (desc->formulation != plan->desc.formulation) return fail(plan, GSM_E_INVALID, "gsm_plan_set_cell: formulation differs");
    if (desc->eps_grid_host) {
        if (!voxel_dims_ok(desc->voxels, desc->orders))
            return fail(plan, GSM_E_INVALID, "voxels[a] must satisfy 2N-1 <= voxels <= 2048");
    } else {
        for (int i = 0; i < desc->n_shapes; ++i)
            if (desc->shapes[i].kind < GSM_SPHERE || desc->shapes[i].kind > GSM_POLYHEDRON)
                return fail(plan, GSM_E_INVALID, "unknown shape kind");
        for (int i = 0; i < desc->n_shapes; ++i)
            if (desc->shapes[i].kind == GSM_POLYHEDRON) {
                ShapeDev q{};
                std::vector<PolyFace> pf;
                std::vector<PolyEdge> pe;
                if (!prepare_polyhedron(desc->shapes[i], q, pf, pe))
                    return fail(plan, GSM_E_INVALID, "malformed polyhedron (indices, degenerate face, or inward orientation)");
            }
    }
    // everything that can be rejected has been: from here on the plan's cell is replaced
    plan->desc.eps_bg_re = desc->eps_bg_re; plan->desc.eps_bg_im = desc->eps_bg_im;
    plan->desc.eps_b_re = desc->eps_b_re;   plan->desc.eps_b_im = desc->eps_b_im;
    plan->desc.n_shapes = desc->n_shapes;   plan->desc.shapes = desc->shapes;
    plan->desc.eps_grid_host = desc->eps_grid_host;
    for (int a = 0; a < 3; ++a) {
        plan->desc.period[a] = desc->period[a];
        plan->desc.voxels[a] = desc->voxels[a];
        plan->geom.K[a] = 2.0 * M_PI / desc->period[a];
    }
    plan->geom.epsb_re = desc->eps_b_re; plan->geom.epsb_im = desc->eps_b_im;
    gsm_status s = build_coeffs(plan);
    if (s == GSM_OK) s = build_spectrum(plan);
    if (s == GSM_OK) {
        cudaError_t e = cudaStreamSynchronize(plan->stream);
        if (e != cudaSuccess) s = fail(plan, GSM_E_CUDA, cudaGetErrorString(e));
    }
    plan->desc.shapes = nullptr;          // caller-owned arrays are not retained
    plan->desc.eps_grid_host = nullptr;
    return s;
}


// ---- retrieval (a10): two-stage scan + pole search -> n_eff, eps_eff -----------------------------------------------
// One stage of the retrieval for many lines at once: line l scans kappa[l][0..n) along dir[l] with amplitude pol[l] at
// k0[l]; ALL points go through ONE gsm_scan.  xi[l][i] = component comp[l] of the 0-th order field, or, for
// comp[l] == -1, its projection on the amplitude, sum_c conj(a_c) E_c / sum_c |a_c|^2 (off-axis directions).
static gsm_status scan_lines(gsm_plan* plan, int nl, const double* dir, const double* pol, const int* comp, const double* k0,
                             const std::vector<double>& kappa, int n, double tol, std::vector<double>& xi, bool* warn) {
    const size_t np = (size_t)nl * n;
    std::vector<double> kb(3 * np), kk(np), pl(6 * np), resp(6 * np);
    for (int l = 0; l < nl; ++l)
        for (int i = 0; i < n; ++i) {
            const size_t p = (size_t)l * n + i;
            for (int a = 0; a < 3; ++a) kb[3 * p + a] = kappa[p] * dir[3 * l + a];
            for (int q = 0; q < 6; ++q) pl[6 * p + q] = pol[6 * l + q];
            kk[p] = k0[l];
        }
    const gsm_status st = gsm_scan(plan, (int)np, kb.data(), kk.data(), pl.data(), tol, resp.data(), nullptr, nullptr, nullptr);
    if (st < 0) return st;
    if (st == GSM_NOT_CONVERGED) *warn = true;
    xi.resize(2 * np);
    for (int l = 0; l < nl; ++l) {
        const double* a = pol + 6 * l;
        const double nrm = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3] + a[4] * a[4] + a[5] * a[5];
        for (int i = 0; i < n; ++i) {
            const size_t p = (size_t)l * n + i;
            if (comp[l] >= 0) {
                xi[2 * p] = resp[6 * p + 2 * comp[l]];
                xi[2 * p + 1] = resp[6 * p + 2 * comp[l] + 1];
            } else {
                double re = 0.0, im = 0.0;
                for (int c = 0; c < 3; ++c) {   // conj(a_c) E_c
                    re += a[2 * c] * resp[6 * p + 2 * c] + a[2 * c + 1] * resp[6 * p + 2 * c + 1];
                    im += a[2 * c] * resp[6 * p + 2 * c + 1] - a[2 * c + 1] * resp[6 * p + 2 * c];
                }
                xi[2 * p] = re / nrm;
                xi[2 * p + 1] = im / nrm;
            }
        }
    }
    return GSM_OK;
}

extern "C" gsm_status gsm_retrieve_neff_many(gsm_plan* plan, int nlines, const double* dir, const double* pol, const int* comp,
                                             const double* k0, const double* n_lo, const double* n_hi, int ncoarse,
                                             int nfine, double fine_step, double tol, double* out, int* line_status) {
    if (!plan) return GSM_E_INVALID;
    const int Np = 5, Nd = 10;
    if (nlines < 0 || !dir || !pol || !comp || !k0 || !n_lo || !n_hi || !out || ncoarse < Np + Nd || nfine < Np + Nd ||
        (nfine & 1) || !(fine_step > 0.0) || !(tol > 0.0))
        return fail(plan, GSM_E_INVALID, "gsm_retrieve_neff: bad argument");
    for (int l = 0; l < nlines; ++l)
        if (comp[l] < -1 || comp[l] > 2 || !(k0[l] > 0.0) || !(n_hi[l] > n_lo[l]))
            return fail(plan, GSM_E_INVALID, "gsm_retrieve_neff: bad argument");
    if (nlines == 0) return GSM_OK;
    bool warn = false, missing = false;
    std::vector<double> kappa((size_t)nlines * ncoarse), xi, eta_c(nlines, 0.0);
    std::vector<int> ok(nlines, 1);
    for (int l = 0; l < nlines; ++l)
        for (int i = 0; i < ncoarse; ++i)
            kappa[(size_t)l * ncoarse + i] = k0[l] * (n_lo[l] + (n_hi[l] - n_lo[l]) * i / (ncoarse - 1));
    gsm_status st = scan_lines(plan, nlines, dir, pol, comp, k0, kappa, ncoarse, tol, xi, &warn);
    if (st < 0) return st;
    double eta[2 * Np], zeta[2 * Np];
    for (int l = 0; l < nlines; ++l) {
        int best = -1;
        const double* kp = kappa.data() + (size_t)l * ncoarse;
        st = gsm_pole_search(ncoarse, kp, xi.data() + 2 * (size_t)l * ncoarse, Np, Nd, kp[0], kp[ncoarse - 1], eta, zeta, &best);
        if (st < 0 || best < 0) { ok[l] = 0; missing = true; eta_c[l] = 0.5 * (kp[0] + kp[ncoarse - 1]); }
        else eta_c[l] = eta[2 * best];
    }
    kappa.assign((size_t)nlines * nfine, 0.0);
    for (int l = 0; l < nlines; ++l)
        for (int i = 0; i < nfine; ++i)      // nfine even: the estimate falls mid-way between the two middle nodes
            kappa[(size_t)l * nfine + i] = eta_c[l] + fine_step * k0[l] * (i - 0.5 * (nfine - 1));
    st = scan_lines(plan, nlines, dir, pol, comp, k0, kappa, nfine, tol, xi, &warn);
    if (st < 0) return st;
    for (int l = 0; l < nlines; ++l) {
        double* o = out + 6 * (size_t)l;
        int best = -1;
        const double* kp = kappa.data() + (size_t)l * nfine;
        if (ok[l]) st = gsm_pole_search(nfine, kp, xi.data() + 2 * (size_t)l * nfine, Np, Nd, kp[0], kp[nfine - 1], eta, zeta, &best);
        if (!ok[l] || st < 0 || best < 0) {
            ok[l] = 0; missing = true;
            for (int q = 0; q < 6; ++q) o[q] = NAN;
        } else {
            const double nr = eta[2 * best] / k0[l], ni = eta[2 * best + 1] / k0[l];
            o[0] = nr; o[1] = ni;
            o[2] = nr * nr - ni * ni; o[3] = 2.0 * nr * ni;
            o[4] = zeta[2 * best]; o[5] = zeta[2 * best + 1];
        }
        if (line_status) line_status[l] = ok[l] ? GSM_OK : GSM_E_INVALID;
    }
    if (missing) return fail(plan, GSM_E_INVALID, "gsm_retrieve_neff: no pole inside the scanned window of at least one line");
    return warn ? GSM_NOT_CONVERGED : GSM_OK;
}

extern "C" gsm_status gsm_retrieve_neff(gsm_plan* plan, const double dir[3], const double pol[6], int comp, double k0,
                                        double n_lo, double n_hi, int ncoarse, int nfine, double fine_step, double tol,
                                        double out[6]) {
    if (!dir || !pol || !out) return plan ? fail(plan, GSM_E_INVALID, "gsm_retrieve_neff: bad argument") : GSM_E_INVALID;
    return gsm_retrieve_neff_many(plan, 1, dir, pol, &comp, &k0, &n_lo, &n_hi, ncoarse, nfine, fine_step, tol, out, nullptr);
}
