// apply_static.cu - gsm_apply_static: the operator y = x - G (T x) of Eq. 4 / Eq. 5 for small cells,
// without a plan and without a single device or pinned-host allocation.
//
// Why it exists.  Everything else in this library works on a gsm_plan, and gsm_plan_create obtains the coefficient
// spectrum, the FFT workspace and the Krylov pool from cudaMalloc.  Some programs that embed the library may not do
// that: a host application whose own allocator (PyTorch's caching allocator, a serving engine's pre-reserved pool, an
// RMM arena) already holds the device's memory, so that a further cudaMalloc fails or bypasses its accounting; a
// process running under a per-client memory limit; a latency-bound loop that cannot afford the device-wide
// synchronisation cudaMalloc / cudaFree imply.  Such a caller owns buffers from its own allocator for the operator's
// inputs (the Toeplitz generator c_d, the field x) and output (y), but has nowhere to put the intermediates - the
// transformed coefficient grid and the z-transformed field W that the three passes of apply.cu exchange through global
// memory.  Here those live in ONE file-scope __device__ array of fixed size that is part of the loaded library image.
//
// What it costs.  GSM_STATIC_SCRATCH_BYTES (about 2.5 MiB) on every GPU that loads the library, held until the process
// exits, whether or not the entry point is ever called.  The fixed size is the reason for the limits GSM_STATIC_MAX_ORDER
// and GSM_STATIC_MAX_BATCH.  The coefficient spectrum is rebuilt on every call (five extra small launches): there is no
// plan to keep it in.
//
// Sharing.  There is one array per device, not per call: every call on a device uses it and it keeps whatever the
// last call left.  Nothing relies on old contents - the circulant grid is cleared (cudaMemsetAsync) before the
// coefficients are scattered into it, and every other region is overwritten in full before it is read - but two calls
// that overlap on the GPU (different streams, or different host threads) race on it.  Serialise them.
//
// The kernels are the generic passes of apply.cu and plan_kernels.cu, unchanged; only the workspace pointers differ.
#include <cmath>
#include <mutex>
#include <string>
#include <vector>

#include "gsm_internal.cuh"

namespace gsm {

// ---- layout of the scratch array, in complex numbers ------------------------------------------------------------
constexpr int kMaxOrder = GSM_STATIC_MAX_ORDER;                 // harmonics per axis
constexpr int kMaxBatch = GSM_STATIC_MAX_BATCH;
constexpr int kMaxP = 32;                                       // FFT points per axis: smallest power of two >= 2 * 16 - 1
constexpr size_t kTwOff = 0;                                    // twiddle tables of P = 1, 2, 4, .. 32 at offset P - 1
constexpr size_t kTwLen = 64;
constexpr size_t kKOff = kTwOff + kTwLen;                       // k_bloch [batch][3] then k0 [batch], as doubles
constexpr size_t kKLen = 16;
constexpr size_t kPadOff = kKOff + kKLen;                       // circulant embedding of c_d, transformed in place
constexpr size_t kPadLen = (size_t)kMaxP * kMaxP * kMaxP;
constexpr size_t kChatOff = kPadOff + kPadLen;                  // coefficient spectrum in the passes' position order
constexpr size_t kChatLen = kPadLen;
constexpr size_t kWOff = kChatOff + kChatLen;                   // W[batch][3][P3][N1 N2]
constexpr size_t kWLen = (size_t)kMaxBatch * 3 * kMaxP * kMaxOrder * kMaxOrder;
constexpr size_t kScratchLen = kWOff + kWLen;
static_assert(kScratchLen * sizeof(cplx) == GSM_STATIC_SCRATCH_BYTES, "gsm.h states the size of the static scratch");
static_assert(kKLen * 2 >= (size_t)kMaxBatch * 4, "wavevector slot too small");

// The scratch itself.  In host code this name is only a handle for cudaGetSymbolAddress / cudaMemcpyToSymbol - it is NOT
// a device address and must never be handed to a kernel; device_setup() asks the runtime for the real address.
static __device__ __align__(256) cplx g_static_scratch[kScratchLen];

constexpr int kMaxDevices = 64;
static std::mutex g_setup_mutex;
static cplx* g_scratch_addr[kMaxDevices] = {};   // device address of g_static_scratch on each device, null = not set up

// Once per device, with that device current: find the array's device address, raise the kernels' shared-memory limits
// and fill the twiddle tables (same values as a plan's: host cos / sin, exact on the axes).  Synchronous copies.
static cudaError_t device_setup(int dev, cplx** out) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (g_scratch_addr[dev]) { *out = g_scratch_addr[dev]; return cudaSuccess; }
    cplx* base = nullptr;
    cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&base), g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!base) return cudaErrorInvalidSymbol;
    e = apply_init_attributes();
    if (e == cudaSuccess) e = plan_init_attributes();
    if (e != cudaSuccess) return e;
    std::vector<double> h(2 * kTwLen, 0.0);
    for (int P = 1; P <= kMaxP; P *= 2) {
        double* t = h.data() + 2 * (P - 1);
        for (int k = 0; k < P; ++k) {
            const double a = -2.0 * M_PI * (double)k / (double)P;
            t[2 * k] = std::cos(a);
            t[2 * k + 1] = std::sin(a);
        }
        if (P >= 2) { t[2 * (P / 2)] = -1.0; t[2 * (P / 2) + 1] = 0.0; }
        if (P >= 4) { t[2 * (P / 4)] = 0.0; t[2 * (P / 4) + 1] = -1.0; t[2 * (3 * P / 4)] = 0.0; t[2 * (3 * P / 4) + 1] = 1.0; }
    }
    e = cudaMemcpy(base + kTwOff, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    g_scratch_addr[dev] = base;
    *out = base;
    return cudaSuccess;
}

// FFT length and radix plan per axis: the same choices gsm_plan_create makes for these sizes, so that a plan and this
// entry point run the identical butterfly network.
static bool axis_for_order(int N, AxisPlan* ax) {
    int P = 1;
    if (N > 1) while (P < 2 * N - 1) P *= 2;
    ax->P = P; ax->N = N; ax->nst = 0;
    for (int i = 0; i < 4; ++i) ax->radix[i] = 1;
    switch (P) {
        case 1: break;
        case 2: ax->nst = 1; ax->radix[0] = 2; break;
        case 4: ax->nst = 1; ax->radix[0] = 4; break;
        case 8: ax->nst = 1; ax->radix[0] = 8; break;
        case 16: ax->nst = 2; ax->radix[0] = 4; ax->radix[1] = 4; break;
        case 32: ax->nst = 2; ax->radix[0] = 4; ax->radix[1] = 8; break;
        default: return false;
    }
    return true;
}

static int odd_up(int v) { return v | 1; }

gsm_status apply_static(const double period[3], const int orders[3], double eps_b_re, double eps_b_im, int formulation,
                        const void* d_coef, int batch, const double* k_bloch, const double* k0, const void* d_x, void* d_y,
                        cudaStream_t st, std::string* err) {
    auto bad = [&](gsm_status s, const std::string& m) { *err = "gsm_apply_static: " + m; return s; };
    if (!period || !orders || !d_coef || !k_bloch || !k0 || !d_x || !d_y) return bad(GSM_E_INVALID, "null argument");
    if (d_x == d_y) return bad(GSM_E_INVALID, "d_x and d_y must not overlap");
    for (int a = 0; a < 3; ++a) {
        if (orders[a] < 1) return bad(GSM_E_INVALID, "orders must be >= 1");
        if (orders[a] > kMaxOrder)
            return bad(GSM_E_INVALID, "orders[" + std::to_string(a) + "] = " + std::to_string(orders[a]) + " exceeds GSM_STATIC_MAX_ORDER = " +
                       std::to_string(kMaxOrder) + " (the fixed static scratch has no room; use a gsm_plan and gsm_apply)");
        if (!(period[a] > 0.0)) return bad(GSM_E_INVALID, "periods must be positive");
    }
    if (batch < 1) return bad(GSM_E_INVALID, "batch must be >= 1");
    if (batch > kMaxBatch)
        return bad(GSM_E_INVALID, "batch = " + std::to_string(batch) + " exceeds GSM_STATIC_MAX_BATCH = " + std::to_string(kMaxBatch) +
                   " (the fixed static scratch has no room; split the call or use a gsm_plan and gsm_apply)");
    if (eps_b_re == 0.0 && eps_b_im == 0.0) return bad(GSM_E_INVALID, "eps_b must be non-zero");
    if (formulation != GSM_FORM_E && formulation != GSM_FORM_H) return bad(GSM_E_INVALID, "formulation must be GSM_FORM_E or GSM_FORM_H");

    ApplyGeom g{};
    g.N1 = orders[0]; g.N2 = orders[1]; g.N3 = orders[2];
    g.NL = g.N1 * g.N2;
    g.n = (long)g.NL * g.N3;
    for (int a = 0; a < 3; ++a) {
        if (!axis_for_order(orders[a], &g.ax[a])) return bad(GSM_E_INVALID, "unsupported FFT size");
        g.K[a] = 2.0 * M_PI / period[a];
        g.mmin[a] = (orders[a] % 2 == 1) ? -(orders[a] - 1) / 2 : -orders[a] / 2;
    }
    g.epsb_re = eps_b_re; g.epsb_im = eps_b_im;
    g.hform = formulation == GSM_FORM_H;
    g.L = g.NL < 32 ? g.NL : 32;
    g.Lst = odd_up(g.L);
    g.RS3 = odd_up(3 * g.L);
    g.N1s = odd_up(g.N1);
    g.CB = g.ax[1].P < 32 ? g.ax[1].P : 32;
    g.CBs = odd_up(g.CB);
    g.YR = g.N1 < 32 ? g.N1 : 32;
    g.YRs = odd_up(g.YR);
    g.split = 0;
    if (apply_smem_max(g) > 227 * 1024) return bad(GSM_E_INVALID, "orders too large for the shared-memory tiles");
    const int P[3] = {g.ax[0].P, g.ax[1].P, g.ax[2].P};
    const size_t np = (size_t)P[0] * P[1] * P[2], nw = (size_t)batch * 3 * P[2] * g.NL;
    if (np > kPadLen || nw > kWLen) return bad(GSM_E_INVALID, "internal: size exceeds the static scratch");

    // eps_b must keep k_m.k_m != k_b^2 for every kept harmonic (same threshold as gsm_apply)
    for (int b = 0; b < batch; ++b) {
        const double kb2r = k0[b] * k0[b] * eps_b_re, kb2i = k0[b] * k0[b] * eps_b_im, mag = std::hypot(kb2r, kb2i);
        double best = INFINITY;
        for (int i1 = 0; i1 < g.N1; ++i1)
            for (int i2 = 0; i2 < g.N2; ++i2)
                for (int i3 = 0; i3 < g.N3; ++i3) {
                    const double k1 = k_bloch[3 * b] + (i1 + g.mmin[0]) * g.K[0], k2 = k_bloch[3 * b + 1] + (i2 + g.mmin[1]) * g.K[1],
                                 k3 = k_bloch[3 * b + 2] + (i3 + g.mmin[2]) * g.K[2];
                    best = std::fmin(best, std::fabs(k1 * k1 + k2 * k2 + k3 * k3 - kb2r));
                }
        const double dist = std::hypot(best, kb2i);
        if (!(dist > 1e-12 * mag) || !std::isfinite(dist)) return bad(GSM_E_SINGULAR_BASIS, "k_m.k_m == k_b^2 for some m");
    }

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return bad(GSM_E_CUDA, std::string("cudaGetDevice failed: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return bad(GSM_E_INVALID, "device ordinal out of range");
    cplx* base = nullptr;
    e = device_setup(dev, &base);
    if (e != cudaSuccess) return bad(GSM_E_CUDA, std::string("set-up of the static scratch failed: ") + cudaGetErrorString(e));

    cplx *pad = base + kPadOff, *chat = base + kChatOff, *W = base + kWOff;
    double* d_kvec = reinterpret_cast<double*>(base + kKOff);
    double* d_k0 = d_kvec + 3 * kMaxBatch;
    for (int a = 0; a < 3; ++a) g.tw[a] = base + kTwOff + (P[a] - 1);
    g.chat = chat;
    auto ck = [&](cudaError_t ce, const char* what) {
        if (ce == cudaSuccess) return true;
        *err = std::string("gsm_apply_static: ") + what + " failed: " + cudaGetErrorString(ce);
        return false;
    };
    if (!ck(cudaMemcpyAsync(d_kvec, k_bloch, sizeof(double) * 3 * batch, cudaMemcpyHostToDevice, st), "copy of k_bloch")) return GSM_E_CUDA;
    if (!ck(cudaMemcpyAsync(d_k0, k0, sizeof(double) * batch, cudaMemcpyHostToDevice, st), "copy of k0")) return GSM_E_CUDA;
    // a0 (second half): Chat = forward network of the circulant embedding of c_d, scaled, in position order.
    // launch_embed clears the grid first - the one region that must start at zero.
    if (!ck(launch_embed(static_cast<const cplx*>(d_coef), orders, P, pad, st), "embed")) return GSM_E_CUDA;
    if (!ck(launch_fft_axis(pad, (long)P[0] * P[1], g.ax[2], 1, g.tw[2], st), "coefficient FFT (z)")) return GSM_E_CUDA;
    if (!ck(launch_fft_axis(pad, (long)P[0], g.ax[1], P[2], g.tw[1], st), "coefficient FFT (y)")) return GSM_E_CUDA;
    if (!ck(launch_fft_axis(pad, 1, g.ax[0], (long)P[1] * P[2], g.tw[0], st), "coefficient FFT (x)")) return GSM_E_CUDA;
    if (!ck(launch_chat_layout(pad, P, chat, st), "spectrum layout")) return GSM_E_CUDA;
    // a1-a5: the three passes, W in the static scratch
    if (!ck(launch_apply(g, batch, d_kvec, d_k0, static_cast<const cplx*>(d_x), static_cast<cplx*>(d_y), W, nullptr, nullptr, st,
                         nullptr, 0.0), "operator apply")) return GSM_E_CUDA;
    return GSM_OK;
}

}  // namespace gsm
