// apply64.cu - operator-apply passes specialised for a 64-point axis (17..32 harmonics kept, e.g. the 31^3 configs of
// BASELINE.json), same data layouts and the same radix-8 x radix-8 network as the generic kernels of apply.cu
// (Toeplitz product by FFT).
//
// Eight lanes share one line: lane u of the group runs butterfly u of both stages with its 8 points in registers.
//   forward  stage 1: inputs e = u + 8p (only p < 4 can be non-zero: the padding half is never loaded or added),
//                     outputs y_q w64^(u q) for e = u + 8q; the 7 twiddles depend on (u, q) only and live in
//                     registers for the whole kernel;
//            exchange: an 8 x 8 transpose inside the group through a warp-private scratch line (padded index
//                     e + e/8, conflict-free both ways) fenced by __syncwarp only;
//            stage 2: inputs e = 8u + p, no twiddles, outputs at positions 8u + q.
//   inverse = mirror image; its last stage forms only the 4 outputs that are kept.
// A 64 x 64 plane therefore needs two block-wide barriers (y <-> x hand-over), not one per stage, no index
// division, and no twiddle traffic.
#include "gsm_internal.cuh"
#include "fft_group.cuh"

namespace gsm {

// ------------------------------------------------------------------------------------------- pass 2, P1 = P2 = 64
// One CTA per (solve b, z-position pos3), 8 warps, the three component planes in turn.  A[r][col]: row r = y-position (64), 32 columns
// = x-index i1 rotated by r/8, so that both the y-phase (lanes differ in u = r/8) and the x-phase (lanes differ in
// i1) touch 8 distinct 16-byte bank groups per quarter-warp.
//   y forward : group (i1 = 4 warp + ln) reads its 4 x 8 inputs straight from W (contiguous in i2), writes rows of A
//   x         : group (row r) reads <= 32 inputs from A, forward, * Chat, inverse, writes the kept 32 back in place
//   y inverse : mirror of y forward, stores straight to W
// chat64 is Chat permuted so that the 8 lanes of a group read 8 consecutive coefficients:
//   chat64[((pos3 * 64 + r) * 8 + q) * 8 + u] = Chat[pos3][pos1 = 8u + q][pos2 = r].
#define XY64_MINB 2   // measured: 2 CTAs/SM at 122 registers (no spills) beats 3 CTAs/SM at 80 (46 vs 52 ms)
__global__ void __launch_bounds__(256, XY64_MINB) xy_conv64_kernel(ApplyGeom g, cplx* __restrict__ W,
                                                           const cplx* __restrict__ chat64,
                                                           const int* __restrict__ active) {
    // one CTA per (solve b, z-position pos3); the three components are done in turn, the inputs of the next component
    // being fetched from W while the current one is transformed
    const int b = blockIdx.y, pos3 = blockIdx.x;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* A = reinterpret_cast<cplx*>(smem_raw);   // [64][32]
    cplx* scratch = A + 64 * 32;                   // [32 lines][SC_LINE]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, u = lane & 7, ln = lane >> 3;
    const int N1 = g.N1, N2 = g.N2;
    cplx tw[7];
    load_group_twiddles(tw, g.tw[0], u);
    cplx* sc = scratch + (warp * 4 + ln) * SC_LINE;
    const long cstride = 64L * g.NL;
    cplx* Wp = W + ((long)b * 3 * 64 + pos3) * g.NL;   // component 0; component c at + c * cstride
    const int i1y = warp * 4 + ln;                      // y-phase line of this group
    cplx a[8], nx[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const int i2 = u + 8 * p;
        nx[p] = (i1y < N1 && i2 < N2) ? Wp[i1y * N2 + i2] : make_double2(0.0, 0.0);
    }
#pragma unroll 1
    for (int c = 0; c < 3; ++c, Wp += cstride) {
        {   // ---- y forward
#pragma unroll
            for (int p = 0; p < 4; ++p) a[p] = nx[p];
            if (c < 2) {
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    const int i2 = u + 8 * p;
                    nx[p] = (i1y < N1 && i2 < N2) ? Wp[cstride + i1y * N2 + i2] : make_double2(0.0, 0.0);
                }
            }
            fwd64_group(a, tw, sc, u);
            const int col = (i1y + u) & 31;
#pragma unroll
            for (int q = 0; q < 8; ++q) A[(8 * u + q) * 32 + col] = a[q];
        }
        __syncthreads();
        // ---- x: forward, multiply by the coefficient spectrum, inverse
#pragma unroll 1
        for (int round = 0; round < 2; ++round) {
            const int r = (round * 8 + warp) * 4 + ln;
            cplx* Ar = A + r * 32;
            const int rot = r >> 3;
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int i1 = u + 8 * p;
                a[p] = (i1 < N1) ? Ar[(i1 + rot) & 31] : make_double2(0.0, 0.0);
            }
            const cplx* cp = chat64 + ((long)(pos3 * 64 + r) * 64) + u;
            fwd64_group(a, tw, sc, u);
#pragma unroll
            for (int q = 0; q < 8; ++q) a[q] = cmul(a[q], __ldg(cp + 8 * q));
            inv64_group(a, tw, sc, u);
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int i1 = u + 8 * p;
                if (i1 < N1) Ar[(i1 + rot) & 31] = a[p];
            }
        }
        __syncthreads();
        {   // ---- y inverse
            const int col = (i1y + u) & 31;
#pragma unroll
            for (int q = 0; q < 8; ++q) a[q] = A[(8 * u + q) * 32 + col];
            inv64_group(a, tw, sc, u);
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int i2 = u + 8 * p;
                if (i1y < N1 && i2 < N2) Wp[i1y * N2 + i2] = a[p];
            }
        }
        __syncthreads();   // A is rewritten by the next component's y-forward
    }
}

// ------------------------------------------------------------------------------------------- pass 1, P3 = 64
// CTA = 32 consecutive z-lines of one (b, c).  Each group loads its line's <= 32 inputs straight from x (contiguous),
// transforms, and drops the 64 outputs into a [pos3][32 lines] tile (columns rotated by pos3/8: conflict-free), which
// is then written to W[b][c][pos3][l] as 512-byte rows.
#define ZF64_MINB 4
template <bool HFORM>
__global__ void __launch_bounds__(256, ZF64_MINB) z_forward64_kernel(ApplyGeom g, const cplx* __restrict__ x,
                                                                     cplx* __restrict__ W, const double* __restrict__ kvec,
                                                                     const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* T = reinterpret_cast<cplx*>(smem_raw);   // [64][32] tile, aliases the scratch lines (barrier in between)
    cplx* scratch = T;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, u = lane & 7, ln = lane >> 3;
    const int N3 = g.N3, NL = g.NL;
    cplx tw[7];
    load_group_twiddles(tw, g.tw[2], u);
    cplx* sc = scratch + (warp * 4 + ln) * SC_LINE;
    const int l0 = blockIdx.x * 32, line = warp * 4 + ln, l = l0 + line;
    x += slot_offset(g, b);
    const cplx* xs = x + ((long)b * 3 + c) * g.n + (long)l * N3;
    cplx a[8];
    if (!HFORM) {
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int i3 = u + 8 * p;
            a[p] = (l < NL && i3 < N3) ? xs[i3] : make_double2(0.0, 0.0);
        }
    } else {   // Eq. 5: the Toeplitz product acts on (k x x); component c needs the two other components of x
        const int c1 = c == 2 ? 0 : c + 1, c2 = c1 == 2 ? 0 : c1 + 1;
        const int i1 = l / g.N2, i2 = l - i1 * g.N2;
        const double kk[3] = {kvec[3 * b + 0] + (i1 + g.mmin[0]) * g.K[0], kvec[3 * b + 1] + (i2 + g.mmin[1]) * g.K[1],
                              kvec[3 * b + 2] + g.mmin[2] * g.K[2]};
        const cplx* x1 = x + ((long)b * 3 + c1) * g.n + (long)l * N3;
        const cplx* x2 = x + ((long)b * 3 + c2) * g.n + (long)l * N3;
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int i3 = u + 8 * p;
            if (l < NL && i3 < N3) {
                const double ka = c1 == 2 ? kk[2] + i3 * g.K[2] : kk[c1], kb = c2 == 2 ? kk[2] + i3 * g.K[2] : kk[c2];
                const cplx v1 = x1[i3], v2 = x2[i3];   // (k x x)_c = k_c1 x_c2 - k_c2 x_c1
                a[p] = make_double2(ka * v2.x - kb * v1.x, ka * v2.y - kb * v1.y);
            } else {
                a[p] = make_double2(0.0, 0.0);
            }
        }
    }
    fwd64_group(a, tw, sc, u);
    __syncthreads();   // every warp is done with its scratch lines: the tile may overwrite them
    const int col = (line + u) & 31;
#pragma unroll
    for (int q = 0; q < 8; ++q) T[(8 * u + q) * 32 + col] = a[q];
    __syncthreads();
    cplx* Wd = W + ((long)b * 3 + c) * 64 * NL + l0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int r = k * 8 + warp;                       // one 512-byte row per warp and step
        const int ll = (lane - (r >> 3)) & 31;            // logical line stored in physical column `lane`
        if (l0 + ll < NL) Wd[(long)r * NL + ll] = T[r * 32 + lane];
    }
}

// ------------------------------------------------------------------------------------------- pass 3, P3 = 64
// CTA = 32 consecutive z-lines, all three components.  The [pos3][32 lines] tiles of W arrive by cp.async (16 bytes
// per request, columns rotated like pass 1), double-buffered over the components; each group inverse-transforms its
// line, keeps the <= 4 x 3 kept outputs in registers and applies the Green dyadic of Eq. 4:
//   y_c = x_c - (k_b^2 F_c - k_c (k.F)) / (k.k - k_b^2),  k = k_inc + m o K  (unconjugated k.k).
static __device__ __forceinline__ void cp_async16(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
static __device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> static __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__global__ void __launch_bounds__(256, 2) z_inverse_green64_kernel(ApplyGeom g, const cplx* __restrict__ W,
                                                                   const cplx* __restrict__ x, cplx* __restrict__ y,
                                                                   const double* __restrict__ kvec,
                                                                   const double* __restrict__ k0s,
                                                                   const int* __restrict__ active) {
    const int b = blockIdx.y;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* T0 = reinterpret_cast<cplx*>(smem_raw);   // two [64][32] tiles
    cplx* T1 = T0 + 64 * 32;
    cplx* scratch = T1 + 64 * 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, u = lane & 7, ln = lane >> 3;
    const int N3 = g.N3, NL = g.NL;
    const int l0 = blockIdx.x * 32, line = warp * 4 + ln, l = l0 + line;
    auto load_tile = [&](cplx* T, int c) {
        const cplx* Ws = W + ((long)b * 3 + c) * 64 * NL + l0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int r = k * 8 + warp;
            const int ll = (lane - (r >> 3)) & 31;
            if (l0 + ll < NL) cp_async16(&T[r * 32 + lane], Ws + (long)r * NL + ll);
        }
        cp_async_commit();
    };
    load_tile(T0, 0);
    load_tile(T1, 1);
    cplx tw[7];
    load_group_twiddles(tw, g.tw[2], u);
    cplx* sc = scratch + (warp * 4 + ln) * SC_LINE;
    const int col = (line + u) & 31;
    cplx F[3][4];
    cplx a[8];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (c < 2) cp_async_wait<1>(); else cp_async_wait<0>();
        __syncthreads();
        const cplx* T = (c & 1) ? T1 : T0;
#pragma unroll
        for (int q = 0; q < 8; ++q) a[q] = T[(8 * u + q) * 32 + col];
        if (c == 0) {           // tile 0 is consumed: refill it with component 2
            __syncthreads();
            load_tile(T0, 2);
        }
        inv64_group(a, tw, sc, u);
#pragma unroll
        for (int p = 0; p < 4; ++p) F[c][p] = a[p];
    }
    if (l >= NL) return;
    const double k0 = k0s[b];
    const double kb2r = k0 * k0 * g.epsb_re, kb2i = k0 * k0 * g.epsb_im;
    const int i1 = l / g.N2, i2 = l - i1 * g.N2;
    const double k1 = kvec[3 * b + 0] + (i1 + g.mmin[0]) * g.K[0];
    const double k2 = kvec[3 * b + 1] + (i2 + g.mmin[1]) * g.K[1];
    const double k12 = k1 * k1 + k2 * k2;
    const long base = (long)b * 3 * g.n + (long)l * N3 + slot_offset(g, b);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const int i3 = u + 8 * p;
        if (i3 >= N3) continue;
        const double k3 = kvec[3 * b + 2] + (i3 + g.mmin[2]) * g.K[2];
        const cplx F0 = F[0][p], F1 = F[1][p], F2 = F[2][p];
        const cplx s = make_double2(k1 * F0.x + k2 * F1.x + k3 * F2.x, k1 * F0.y + k2 * F1.y + k3 * F2.y);
        const double dr = k12 + k3 * k3 - kb2r, di = -kb2i;
        const double inv = 1.0 / (dr * dr + di * di);
        const cplx rden = make_double2(dr * inv, -di * inv);   // 1 / (k.k - k_b^2)
        const cplx kb2 = make_double2(kb2r, kb2i);
        const double kk[3] = {k1, k2, k3};
        const cplx Fc[3] = {F0, F1, F2};
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            cplx num;
            if (g.hform) {   // Eq. 5: y = x + (k x F) / (k.k - k_b^2)
                const int c1 = c == 2 ? 0 : c + 1, c2 = c1 == 2 ? 0 : c1 + 1;
                num = make_double2(-(kk[c1] * Fc[c2].x - kk[c2] * Fc[c1].x), -(kk[c1] * Fc[c2].y - kk[c2] * Fc[c1].y));
            } else {
                num = cmul(kb2, Fc[c]);
                num.x -= kk[c] * s.x;
                num.y -= kk[c] * s.y;
            }
            const cplx q = cmul(num, rden);
            const cplx xv = x[base + c * g.n + i3];
            y[base + c * g.n + i3] = make_double2(xv.x - q.x, xv.y - q.y);
        }
    }
}

__global__ void chat64_layout_kernel(const cplx* __restrict__ chat, cplx* __restrict__ chat64) {
    const long total = 64L * 64 * 64;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int u = (int)(i & 7), q = (int)((i >> 3) & 7), r = (int)((i >> 6) & 63), p3 = (int)(i >> 12);
        chat64[i] = chat[((long)p3 * 64 + (8 * u + q)) * 64 + r];
    }
}

static const size_t XY64_SMEM = sizeof(cplx) * (64 * 32 + 32 * SC_LINE);

bool apply64_usable(const ApplyGeom& g) {
    return g.ax[0].P == 64 && g.ax[1].P == 64 && g.ax[2].P == 64 && g.N1 <= 32 && g.N2 <= 32 && g.N3 <= 32;
}
cudaError_t launch_chat64_layout(const cplx* d_chat, cplx* d_chat64, cudaStream_t st) {
    chat64_layout_kernel<<<1024, 256, 0, st>>>(d_chat, d_chat64);
    return cudaGetLastError();
}
cudaError_t launch_xy_conv64(const ApplyGeom& g, int batch, cplx* d_W, const cplx* d_chat64, const int* d_active,
                             cudaStream_t st) {
    xy_conv64_kernel<<<dim3(64, batch), 256, XY64_SMEM, st>>>(g, d_W, d_chat64, d_active);
    return cudaGetLastError();
}
static const size_t ZF64_SMEM = sizeof(cplx) * (32 * SC_LINE);   // >= 64 * 32 tile
static const size_t ZI64_SMEM = sizeof(cplx) * (2 * 64 * 32 + 32 * SC_LINE);
cudaError_t launch_z_forward64(const ApplyGeom& g, int batch, const cplx* d_x, cplx* d_W, const double* d_kvec,
                               const int* d_active, cudaStream_t st) {
    const dim3 grid((g.NL + 31) / 32, 3, batch);
    if (g.hform) z_forward64_kernel<true><<<grid, 256, ZF64_SMEM, st>>>(g, d_x, d_W, d_kvec, d_active);
    else z_forward64_kernel<false><<<grid, 256, ZF64_SMEM, st>>>(g, d_x, d_W, d_kvec, d_active);
    return cudaGetLastError();
}
cudaError_t launch_z_inverse_green64(const ApplyGeom& g, int batch, const cplx* d_W, const cplx* d_x, cplx* d_y,
                                     const double* d_kvec, const double* d_k0, const int* d_active, cudaStream_t st) {
    z_inverse_green64_kernel<<<dim3((g.NL + 31) / 32, batch), 256, ZI64_SMEM, st>>>(g, d_W, d_x, d_y, d_kvec, d_k0,
                                                                                     d_active);
    return cudaGetLastError();
}
cudaError_t apply64_init_attributes() {
    cudaError_t e = cudaFuncSetAttribute(xy_conv64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XY64_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(z_forward64_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZF64_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(z_forward64_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZF64_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(z_inverse_green64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ZI64_SMEM);
    return e;
}

}  // namespace gsm
