// apply.cu - the GSM operator y = x - G (T x) of Eq. 4 as three fused passes, complex fp64.
//
// (T x)_{c,m} = sum_m' c_{m-m'} x_{c,m'} is a 3-D Toeplitz product done by circulant embedding in a
// P1 x P2 x P3 grid.  The zero padding is never stored and only the N^3 needed outputs are produced:
//
//   pass 1  z_forward   x[b][c][l][i3] --z-FFT (N3 valid in, P3 out)--> W[b][c][pos3][l]          l = i1*N2+i2
//   pass 2  xy_conv     per (b,c,pos3): plane W[.][l] -> y-FFT -> x-FFT -> * Chat -> x-IFFT -> y-IFFT -> W (in place)
//   pass 3  z_inverse   W[b][.][pos3][l] --z-IFFT (N3 valid out)--> F, then the Green dyadic of Eq. 4:
//                       y_c = x_c - (k_b^2 F_c - k_c (k.F)) / (k.k - k_b^2)
//
// The intermediate W is only 2x (not 8x) the field: it is transformed along z alone.  Pass 2 keeps its plane in
// shared memory pruned to N1 rows and expands along x one column batch at a time through a scratch tile, so a
// 128 x 128 plane never has to exist.  FFT outputs stay in the digit-reversed "position" order of fft_device.cuh;
// Chat is stored in the same order, [pos3][pos1][pos2], so the pass-2 read of Chat is contiguous along pos2.
#include "gsm_internal.cuh"

namespace gsm {

static __device__ __forceinline__ void load_tw(cplx* dst, const cplx* __restrict__ src, int P) {
    for (int i = threadIdx.x; i < P; i += blockDim.x) dst[i] = src[i];
}

// ---------------------------------------------------------------------------------------------------- pass 1
// Eq. 5 (H-form): the Toeplitz product acts on (k_m x x_m); component c of that cross product
static __device__ __forceinline__ cplx cross_k_comp(int c, double k1, double k2, double k3, cplx x0, cplx x1, cplx x2) {
    if (c == 0) return make_double2(k2 * x2.x - k3 * x1.x, k2 * x2.y - k3 * x1.y);
    if (c == 1) return make_double2(k3 * x0.x - k1 * x2.x, k3 * x0.y - k1 * x2.y);
    return make_double2(k1 * x1.x - k2 * x0.x, k1 * x1.y - k2 * x0.y);
}

__global__ void __launch_bounds__(256) z_forward_kernel(ApplyGeom g, const cplx* __restrict__ x, cplx* __restrict__ W,
                                                        const double* __restrict__ kvec,
                                                        const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);
    cplx* S = tw + g.ax[2].P;
    const int P3 = g.ax[2].P, N3 = g.N3;
    const int l0 = blockIdx.x * g.L;
    const int nl = min(g.L, g.NL - l0);
    load_tw(tw, g.tw[2], P3);
    x += slot_offset(g, b);
    const cplx* xs = x + ((long)b * 3 + c) * g.n + (long)l0 * N3;
    if (!g.hform) {
        for (int i = threadIdx.x; i < nl * N3; i += blockDim.x) {
            const int l = i / N3, i3 = i - l * N3;
            S[i3 * g.Lst + l] = xs[i];
        }
    } else {
        const cplx* xb = x + (long)b * 3 * g.n + (long)l0 * N3;
        for (int i = threadIdx.x; i < nl * N3; i += blockDim.x) {
            const int l = i / N3, i3 = i - l * N3;
            const int lg = l0 + l, i1 = lg / g.N2, i2 = lg - i1 * g.N2;
            const double k1 = kvec[3 * b + 0] + (i1 + g.mmin[0]) * g.K[0];
            const double k2 = kvec[3 * b + 1] + (i2 + g.mmin[1]) * g.K[1];
            const double k3 = kvec[3 * b + 2] + (i3 + g.mmin[2]) * g.K[2];
            S[i3 * g.Lst + l] = cross_k_comp(c, k1, k2, k3, xb[i], xb[g.n + i], xb[2 * g.n + i]);
        }
    }
    __syncthreads();
    fft_forward(g.ax[2], Lines{S, g.Lst, 1}, nl, tw, N3);
    cplx* Wd = W + ((long)b * 3 + c) * P3 * g.NL + l0;
    for (int i = threadIdx.x; i < nl * P3; i += blockDim.x) {
        const int pos = i / nl, l = i - pos * nl;
        Wd[(long)pos * g.NL + l] = S[pos * g.Lst + l];
    }
}

// ---------------------------------------------------------------------------------------------------- pass 2
__global__ void __launch_bounds__(256) xy_conv_kernel(ApplyGeom g, cplx* __restrict__ W, const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y, pos3 = blockIdx.x;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P1 = g.ax[0].P, P2 = g.ax[1].P, N1 = g.N1, N2 = g.N2;
    cplx* tw1 = reinterpret_cast<cplx*>(smem_raw);
    cplx* tw2 = tw1 + P1;
    cplx* A = tw2 + P2;                // [P2][N1s]: A[k2 * N1s + i1]
    cplx* B = A + (long)P2 * g.N1s;    // [P1][CBs]: B[k1 * CBs + col]
    load_tw(tw1, g.tw[0], P1);
    load_tw(tw2, g.tw[1], P2);
    cplx* Wp = W + (((long)b * 3 + c) * g.ax[2].P + pos3) * g.NL;
    for (int i = threadIdx.x; i < g.NL; i += blockDim.x) {
        const int i1 = i / N2, i2 = i - i1 * N2;
        A[i2 * g.N1s + i1] = Wp[i];
    }
    __syncthreads();
    // y: N1 lines (index i1, contiguous), elements along k2 at stride N1s
    fft_forward(g.ax[1], Lines{A, g.N1s, 1}, N1, tw2, N2);
    // x: P2 lines (index k2, odd stride N1s), elements along i1 contiguous; CB columns at a time
    const AxisPlan& ax = g.ax[0];
    const cplx* chat = g.chat + (long)pos3 * P1 * P2;
    for (int cb0 = 0; cb0 < P2; cb0 += g.CB) {
        const int ncol = min(g.CB, P2 - cb0);
        const Lines a{A + (long)cb0 * g.N1s, 1, g.N1s};
        const Lines bb{B, g.CBs, 1};
        if (ax.nst == 0) {
            for (int i = threadIdx.x; i < ncol; i += blockDim.x)
                a.p[i * a.ls] = cmul(a.p[i * a.ls], __ldg(chat + cb0 + i));
            __syncthreads();
            continue;
        }
        int Ls = P1;
        for (int s = 0; s + 1 < ax.nst; ++s) {
            dif_stage_rt(ax.radix[s], s == 0 ? a : bb, bb, ncol, P1, Ls, tw1, s == 0 ? N1 : P1);
            Ls /= ax.radix[s];
            __syncthreads();
        }
        const bool only = ax.nst == 1;
        mid_stage_rt(ax.radix[ax.nst - 1], only ? a : bb, only ? a : bb, ncol, P1, chat + cb0, P2, 1, only ? N1 : P1,
                     only ? N1 : P1);
        __syncthreads();
        for (int s = ax.nst - 2; s >= 0; --s) {
            Ls *= ax.radix[s];
            dit_stage_rt(ax.radix[s], bb, s == 0 ? a : bb, ncol, P1, Ls, tw1, s == 0 ? N1 : P1);
            __syncthreads();
        }
    }
    fft_inverse(g.ax[1], Lines{A, g.N1s, 1}, N1, tw2, N2);
    for (int i = threadIdx.x; i < g.NL; i += blockDim.x) {
        const int i1 = i / N2, i2 = i - i1 * N2;
        Wp[i] = A[i2 * g.N1s + i1];
    }
}

// ------------------------------------------------------------------------------ pass 2, split (65..128 harmonics)
// A 256 x 256 plane pruned to 128 rows is 528 KB: it does not fit one SM.  The plane convolution then runs as three
// kernels through the global workspace Y[b][c][pos3][i1][pos2] (expanded along y only, 2 |W|):
//   y_expand   W[i1][i2] --y-FFT (N2 valid in, P2 out)--> Y[i1][pos2]                 rows of i1, YR per CTA
//   x_conv     Y[.][pos2]: x-FFT (N1 valid in) -> * Chat -> x-IFFT (N1 kept), in place    CB columns of pos2 per CTA
//   y_contract Y[i1][pos2] --y-IFFT (N2 kept)--> W[i1][i2]
// Same butterfly network and position order as the single-kernel pass; lanes run along the contiguous index.
__global__ void __launch_bounds__(256) y_expand_kernel(ApplyGeom g, const cplx* __restrict__ W, const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y / g.ax[2].P, pos3 = blockIdx.y - c * g.ax[2].P;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P2 = g.ax[1].P, N2 = g.N2;
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);
    cplx* T = tw + P2;                 // T[k2 * YRs + row]
    const int r0 = blockIdx.x * g.YR, nr = min(g.YR, g.N1 - r0);
    load_tw(tw, g.tw[1], P2);
    const long plane = ((long)b * 3 + c) * g.ax[2].P + pos3;
    const cplx* Wp = W + plane * g.NL + (long)r0 * N2;
    for (int i = threadIdx.x; i < nr * N2; i += blockDim.x) {
        const int r = i / N2, i2 = i - r * N2;
        T[i2 * g.YRs + r] = Wp[i];
    }
    __syncthreads();
    fft_forward(g.ax[1], Lines{T, g.YRs, 1}, nr, tw, N2);
    cplx* Yp = g.Y + (plane * g.N1 + r0) * P2;
    for (int i = threadIdx.x; i < nr * P2; i += blockDim.x) {
        const int r = i / P2, p2 = i - r * P2;
        Yp[(long)r * P2 + p2] = T[p2 * g.YRs + r];
    }
}

__global__ void __launch_bounds__(256) x_conv_kernel(ApplyGeom g, const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y / g.ax[2].P, pos3 = blockIdx.y - c * g.ax[2].P;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P1 = g.ax[0].P, P2 = g.ax[1].P, N1 = g.N1;
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);
    cplx* B = tw + P1;                 // B[k1 * CBs + col]
    const int cb0 = blockIdx.x * g.CB, ncol = min(g.CB, P2 - cb0);
    load_tw(tw, g.tw[0], P1);
    cplx* Yp = g.Y + (((long)b * 3 + c) * g.ax[2].P + pos3) * N1 * P2 + cb0;
    for (int i = threadIdx.x; i < N1 * ncol; i += blockDim.x) {
        const int i1 = i / ncol, col = i - i1 * ncol;
        B[i1 * g.CBs + col] = Yp[(long)i1 * P2 + col];
    }
    __syncthreads();
    const AxisPlan& ax = g.ax[0];
    const cplx* chat = g.chat + (long)pos3 * P1 * P2 + cb0;
    const Lines bb{B, g.CBs, 1};
    int Ls = P1;
    for (int s = 0; s + 1 < ax.nst; ++s) {
        dif_stage_rt(ax.radix[s], bb, bb, ncol, P1, Ls, tw, s == 0 ? N1 : P1);
        Ls /= ax.radix[s];
        __syncthreads();
    }
    const bool only = ax.nst == 1;
    mid_stage_rt(ax.radix[ax.nst - 1], bb, bb, ncol, P1, chat, P2, 1, only ? N1 : P1, only ? N1 : P1);
    __syncthreads();
    for (int s = ax.nst - 2; s >= 0; --s) {
        Ls *= ax.radix[s];
        dit_stage_rt(ax.radix[s], bb, bb, ncol, P1, Ls, tw, s == 0 ? N1 : P1);
        __syncthreads();
    }
    for (int i = threadIdx.x; i < N1 * ncol; i += blockDim.x) {
        const int i1 = i / ncol, col = i - i1 * ncol;
        Yp[(long)i1 * P2 + col] = B[i1 * g.CBs + col];
    }
}

__global__ void __launch_bounds__(256) y_contract_kernel(ApplyGeom g, cplx* __restrict__ W, const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y / g.ax[2].P, pos3 = blockIdx.y - c * g.ax[2].P;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P2 = g.ax[1].P, N2 = g.N2;
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);
    cplx* T = tw + P2;
    const int r0 = blockIdx.x * g.YR, nr = min(g.YR, g.N1 - r0);
    load_tw(tw, g.tw[1], P2);
    const long plane = ((long)b * 3 + c) * g.ax[2].P + pos3;
    const cplx* Yp = g.Y + (plane * g.N1 + r0) * P2;
    for (int i = threadIdx.x; i < nr * P2; i += blockDim.x) {
        const int r = i / P2, p2 = i - r * P2;
        T[p2 * g.YRs + r] = Yp[(long)r * P2 + p2];
    }
    __syncthreads();
    fft_inverse(g.ax[1], Lines{T, g.YRs, 1}, nr, tw, N2);
    cplx* Wp = W + plane * g.NL + (long)r0 * N2;
    for (int i = threadIdx.x; i < nr * N2; i += blockDim.x) {
        const int r = i / N2, i2 = i - r * N2;
        Wp[i] = T[i2 * g.YRs + r];
    }
}

// ---------------------------------------------------------------------------------------------------- pass 3
__global__ void __launch_bounds__(256) z_inverse_green_kernel(ApplyGeom g, const cplx* __restrict__ W,
                                                              const cplx* __restrict__ x, cplx* __restrict__ y,
                                                              const double* __restrict__ kvec,
                                                              const double* __restrict__ k0s,
                                                              const int* __restrict__ active) {
    const int b = blockIdx.y;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P3 = g.ax[2].P, N3 = g.N3;
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);
    cplx* S = tw + P3;                 // [P3][RS3]: S[pos * RS3 + c * nl + l]
    const int l0 = blockIdx.x * g.L;
    const int nl = min(g.L, g.NL - l0);
    load_tw(tw, g.tw[2], P3);
    for (int c = 0; c < 3; ++c) {
        const cplx* Ws = W + ((long)b * 3 + c) * P3 * g.NL + l0;
        for (int i = threadIdx.x; i < nl * P3; i += blockDim.x) {
            const int pos = i / nl, l = i - pos * nl;
            S[pos * g.RS3 + c * nl + l] = Ws[(long)pos * g.NL + l];
        }
    }
    __syncthreads();
    fft_inverse(g.ax[2], Lines{S, g.RS3, 1}, 3 * nl, tw, N3);
    // Green dyadic: k_m = k_inc + m o K, k_b^2 = k0^2 eps_b, unconjugated k.k
    const double kx0 = kvec[3 * b + 0], ky0 = kvec[3 * b + 1], kz0 = kvec[3 * b + 2], k0 = k0s[b];
    const double kb2r = k0 * k0 * g.epsb_re, kb2i = k0 * k0 * g.epsb_im;
    const long base = (long)b * 3 * g.n + (long)l0 * N3 + slot_offset(g, b);
    for (int i = threadIdx.x; i < nl * N3; i += blockDim.x) {
        const int l = i / N3, i3 = i - l * N3;
        const int lg = l0 + l, i1 = lg / g.N2, i2 = lg - i1 * g.N2;
        const double k1 = kx0 + (i1 + g.mmin[0]) * g.K[0];
        const double k2 = ky0 + (i2 + g.mmin[1]) * g.K[1];
        const double k3 = kz0 + (i3 + g.mmin[2]) * g.K[2];
        const cplx F0 = S[i3 * g.RS3 + l], F1 = S[i3 * g.RS3 + nl + l], F2 = S[i3 * g.RS3 + 2 * nl + l];
        const cplx s = make_double2(k1 * F0.x + k2 * F1.x + k3 * F2.x, k1 * F0.y + k2 * F1.y + k3 * F2.y);
        const double dr = k1 * k1 + k2 * k2 + k3 * k3 - kb2r, di = -kb2i;
        const double inv = 1.0 / (dr * dr + di * di);
        const cplx rden = make_double2(dr * inv, -di * inv);   // 1 / (k.k - k_b^2)
        const cplx kb2 = make_double2(kb2r, kb2i);
        const cplx F[3] = {F0, F1, F2};
        const double kk[3] = {k1, k2, k3};
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            cplx num;
            if (g.hform) {   // Eq. 5: y = x - k x F / (k_b^2 - k.k) = x + (k x F) / (k.k - k_b^2)
                const cplx t = cross_k_comp(c, k1, k2, k3, F0, F1, F2);
                num = make_double2(-t.x, -t.y);
            } else {
                num = cmul(kb2, F[c]);
                num.x -= kk[c] * s.x;
                num.y -= kk[c] * s.y;
            }
            const cplx q = cmul(num, rden);
            const cplx xv = x[base + c * g.n + i];
            y[base + c * g.n + i] = make_double2(xv.x - q.x, xv.y - q.y);
        }
    }
}

static size_t smem_pass1(const ApplyGeom& g) { return sizeof(cplx) * ((size_t)g.ax[2].P + (size_t)g.ax[2].P * g.Lst); }
static size_t smem_pass2(const ApplyGeom& g) {
    return sizeof(cplx) * ((size_t)g.ax[0].P + g.ax[1].P + (size_t)g.ax[1].P * g.N1s + (size_t)g.ax[0].P * g.CBs);
}
static size_t smem_pass3(const ApplyGeom& g) { return sizeof(cplx) * ((size_t)g.ax[2].P + (size_t)g.ax[2].P * g.RS3); }
static size_t smem_ypass(const ApplyGeom& g) { return sizeof(cplx) * ((size_t)g.ax[1].P + (size_t)g.ax[1].P * g.YRs); }
static size_t smem_xpass(const ApplyGeom& g) { return sizeof(cplx) * ((size_t)g.ax[0].P + (size_t)g.ax[0].P * g.CBs); }

size_t apply_smem_plane(const ApplyGeom& g) { return smem_pass2(g); }
size_t apply_smem_max(const ApplyGeom& g) {
    size_t m = smem_pass1(g);
    if (g.split) {
        if (smem_ypass(g) > m) m = smem_ypass(g);
        if (smem_xpass(g) > m) m = smem_xpass(g);
    } else if (smem_pass2(g) > m) m = smem_pass2(g);
    if (smem_pass3(g) > m) m = smem_pass3(g);
    return m;
}

// algorithmic bytes of one solve-apply as designed: field vector V = 3n, z-transformed intermediate W_b = 3 P3 NL.
// three launches: z_forward V + W_b, xy_conv 2 W_b, z_inverse_green W_b + 2 V; fused persistent launch: 2 V (W stays in L2).
void bill_apply(const ApplyGeom& g, bool fused, Profiler* prof, double units) {
    if (!prof || units <= 0.0) return;
    const double V = 16.0 * 3.0 * g.n, Wb = 16.0 * 3.0 * g.ax[2].P * g.NL;
    if (fused) {
        prof->bytes[KC_APPLY_FUSED] += 2.0 * V * units;
    } else {
        prof->bytes[KC_Z_FORWARD] += (V + Wb) * units;
        // split path: W -> Y, Y in place, Y -> W with |Y| = 3 P3 N1 P2 complex numbers
        const double Yb = 16.0 * 3.0 * g.ax[2].P * g.N1 * g.ax[1].P;
        prof->bytes[KC_XY_CONV] += (g.split ? 2.0 * Wb + 4.0 * Yb : 2.0 * Wb) * units;
        prof->bytes[KC_Z_INVERSE_GREEN] += (Wb + 2.0 * V) * units;
    }
}

cudaError_t launch_apply(const ApplyGeom& g, int batch, const double* d_kvec, const double* d_k0, const cplx* d_x,
                         cplx* d_y, cplx* d_W, const Fused64Dev* fused, const int* d_active, cudaStream_t st,
                         Profiler* prof, double units) {
    const double Cb = 16.0 * g.ax[0].P * g.ax[1].P * g.ax[2].P;   // the coefficient spectrum is read once per launch
    cudaError_t e = cudaSuccess;
    if (fused && fused->ring) {
        bill_apply(g, true, prof, units);
        ProfScope ps_(prof, KC_APPLY_FUSED, st, Cb);
        return launch_apply_fused64(g, batch, d_kvec, d_k0, d_x, d_y, d_active, *fused, st);
    }
    bill_apply(g, false, prof, units);
    const int nlt = (g.NL + g.L - 1) / g.L;
    { ProfScope ps_(prof, KC_Z_FORWARD, st);
      if (g.chat64) e = launch_z_forward64(g, batch, d_x, d_W, d_kvec, d_active, st);
      else { z_forward_kernel<<<dim3(nlt, 3, batch), 256, smem_pass1(g), st>>>(g, d_x, d_W, d_kvec, d_active); e = cudaGetLastError(); } }
    if (e != cudaSuccess) return e;
    { ProfScope ps_(prof, KC_XY_CONV, st, Cb);
      if (g.chat64) e = launch_xy_conv64(g, batch, d_W, g.chat64, d_active, st);
      else if (g.chat128) e = launch_xy_conv128(g, batch, d_W, g.chat128, d_active, st);
      else if (g.split) {
          const dim3 gy((g.N1 + g.YR - 1) / g.YR, 3 * g.ax[2].P, batch), gx((g.ax[1].P + g.CB - 1) / g.CB, 3 * g.ax[2].P, batch);
          y_expand_kernel<<<gy, 256, smem_ypass(g), st>>>(g, d_W, d_active);
          x_conv_kernel<<<gx, 256, smem_xpass(g), st>>>(g, d_active);
          y_contract_kernel<<<gy, 256, smem_ypass(g), st>>>(g, d_W, d_active);
          e = cudaGetLastError();
      } else { xy_conv_kernel<<<dim3(g.ax[2].P, 3, batch), 256, smem_pass2(g), st>>>(g, d_W, d_active); e = cudaGetLastError(); } }
    if (e != cudaSuccess) return e;
    { ProfScope ps_(prof, KC_Z_INVERSE_GREEN, st);
      if (g.chat64) e = launch_z_inverse_green64(g, batch, d_W, d_x, d_y, d_kvec, d_k0, d_active, st);
      else { z_inverse_green_kernel<<<dim3(nlt, batch), 256, smem_pass3(g), st>>>(g, d_W, d_x, d_y, d_kvec, d_k0, d_active); e = cudaGetLastError(); } }
    return e;
}

}  // namespace gsm

namespace gsm {
cudaError_t apply_init_attributes() {
    cudaError_t e = cudaFuncSetAttribute(z_forward_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(xy_conv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(z_inverse_green_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(y_expand_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(x_conv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(y_contract_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) e = apply64_init_attributes();
    if (e == cudaSuccess) e = apply128_init_attributes();
    return e;
}
}  // namespace gsm
