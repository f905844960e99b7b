// fft_device.cuh - complex-fp64 line FFTs in shared memory for the Toeplitz product of Eq. 4.
//
// Design (sm_100a; plain fp64 ALUs, no tensor cores - the path is not a dense contraction):
//   * A CTA owns a tile of many lines in shared memory.  One thread does one radix-R butterfly (R in {2,4,8})
//     with its R points in registers; stages exchange through shared memory.
//   * Lines are laid out so that consecutive lanes touch consecutive *lines* (line stride 1 or odd in 16-byte
//     units), which makes every 128-bit access conflict-free whatever the butterfly span, and makes the twiddle
//     lookup a broadcast.
//   * Forward = decimation in frequency, natural order in, digit-reversed "position" order out, NO reordering
//     pass.  Inverse = the same network run backwards (decimation in time, conjugate twiddles), positions in,
//     natural order out.  The coefficient spectrum is produced by the same forward network, so it lives in
//     position order too and the permutation never has to be undone on the hot path.
//   * Pruning: the field occupies the first N <= P/2 entries of a length-P line (zero padding of the circulant
//     embedding) and only the first N outputs are needed.  The first forward stage takes `nvalid` and reads zeros
//     beyond it (the padding is never stored); the last inverse stage stores only entries < nvalid.
//   * Twiddles exp(-2 pi i k / P) come from an fp64 table computed on the host (parity budget 1e-9 leaves no room
//     for fast-math sincos).
#pragma once
#include <cuda_runtime.h>

namespace gsm {

typedef double2 cplx;

__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {   // a * conj(b)
    return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y));
}
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx c) {   // a*b + c
    return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
// multiply by -i (forward) or +i (inverse)
template <bool INV> __device__ __forceinline__ cplx mul_mi(cplx a) {
    return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}

#define GSM_SQRT1_2 0.70710678118654752440

// y_q = sum_p a_p exp(-/+ 2 pi i p q / R), in place.
template <int R, bool INV> struct Bfly;

template <bool INV> struct Bfly<2, INV> {
    static __device__ __forceinline__ void run(cplx* a) {
        cplx t = a[0];
        a[0] = cadd(t, a[1]);
        a[1] = csub(t, a[1]);
    }
};

template <bool INV> struct Bfly<4, INV> {
    static __device__ __forceinline__ void run(cplx* a) {
        cplx t0 = cadd(a[0], a[2]), t1 = csub(a[0], a[2]);
        cplx t2 = cadd(a[1], a[3]), t3 = mul_mi<INV>(csub(a[1], a[3]));
        a[0] = cadd(t0, t2);
        a[2] = csub(t0, t2);
        a[1] = cadd(t1, t3);
        a[3] = csub(t1, t3);
    }
};

template <bool INV> struct Bfly<8, INV> {
    static __device__ __forceinline__ void run(cplx* a) {
        cplx e[4] = {a[0], a[2], a[4], a[6]};
        cplx o[4] = {a[1], a[3], a[5], a[7]};
        Bfly<4, INV>::run(e);
        Bfly<4, INV>::run(o);
        // o[k] *= w8^k  (forward w8 = exp(-i pi/4); inverse its conjugate)
        cplx o1, o3;
        if (INV) {
            o1 = make_double2((o[1].x - o[1].y) * GSM_SQRT1_2, (o[1].y + o[1].x) * GSM_SQRT1_2);
            o3 = make_double2((-o[3].x - o[3].y) * GSM_SQRT1_2, (o[3].x - o[3].y) * GSM_SQRT1_2);
        } else {
            o1 = make_double2((o[1].x + o[1].y) * GSM_SQRT1_2, (o[1].y - o[1].x) * GSM_SQRT1_2);
            o3 = make_double2((o[3].y - o[3].x) * GSM_SQRT1_2, (-o[3].x - o[3].y) * GSM_SQRT1_2);
        }
        cplx o2 = mul_mi<INV>(o[2]);
        a[0] = cadd(e[0], o[0]);  a[4] = csub(e[0], o[0]);
        a[1] = cadd(e[1], o1);    a[5] = csub(e[1], o1);
        a[2] = cadd(e[2], o2);    a[6] = csub(e[2], o2);
        a[3] = cadd(e[3], o3);    a[7] = csub(e[3], o3);
    }
};

// Radix plan of one axis: P = prod radix[s]; forward stage s works on sub-transforms of length Ls = P / prod_{t<s}.
struct AxisPlan {
    int P;         // transform length (power of two, 1 = axis not transformed)
    int nst;       // number of stages
    int radix[4];  // radix of forward stage s
    int N;         // harmonics kept along this axis (valid inputs / outputs)
};

// A set of lines in (shared) memory: element e of line l lives at p[l * ls + e * es].
struct Lines {
    cplx* p;
    int es, ls;
};

__device__ __forceinline__ int ilog2(int v) { return 31 - __clz(v); }

// Forward (DIF) stage with sub-transform length Ls on `nlines` lines: butterfly u of a line takes the points
// e_p = block*Ls + pos + p*Ls/R and leaves y_q * w_Ls^(pos q) at e_q.  Inputs with e_p >= nvalid read as zero.
template <int R>
__device__ __forceinline__ void dif_stage(Lines src, Lines dst, int nlines, int P, int Ls, const cplx* __restrict__ tw,
                                          int nvalid) {
    const int sub = Ls / R, lsub = ilog2(sub), nb = P / R, tstep = P / Ls;
    const int total = nlines * nb;
    for (int w = threadIdx.x; w < total; w += blockDim.x) {
        const int u = w / nlines, line = w - u * nlines;
        const int block = u >> lsub, pos = u & (sub - 1);
        const int e0 = block * Ls + pos;
        cplx a[R];
        const cplx* s = src.p + line * src.ls;
#pragma unroll
        for (int p = 0; p < R; ++p) {
            const int e = e0 + p * sub;
            a[p] = (e < nvalid) ? s[e * src.es] : make_double2(0.0, 0.0);
        }
        Bfly<R, false>::run(a);
        cplx* d = dst.p + line * dst.ls;
        d[e0 * dst.es] = a[0];
#pragma unroll
        for (int q = 1; q < R; ++q) {
            const cplx t = tw[pos * q * tstep];
            d[(e0 + q * sub) * dst.es] = (sub > 1) ? cmul(a[q], t) : a[q];
        }
    }
}

// Inverse (DIT) stage: the exact reverse of dif_stage.  Outputs with e_p >= nvalid are not stored.
template <int R>
__device__ __forceinline__ void dit_stage(Lines src, Lines dst, int nlines, int P, int Ls, const cplx* __restrict__ tw,
                                          int nvalid) {
    const int sub = Ls / R, lsub = ilog2(sub), nb = P / R, tstep = P / Ls;
    const int total = nlines * nb;
    for (int w = threadIdx.x; w < total; w += blockDim.x) {
        const int u = w / nlines, line = w - u * nlines;
        const int block = u >> lsub, pos = u & (sub - 1);
        const int e0 = block * Ls + pos;
        cplx a[R];
        const cplx* s = src.p + line * src.ls;
        a[0] = s[e0 * src.es];
#pragma unroll
        for (int q = 1; q < R; ++q) {
            const cplx v = s[(e0 + q * sub) * src.es];
            a[q] = (sub > 1) ? cmulc(v, tw[pos * q * tstep]) : v;
        }
        Bfly<R, true>::run(a);
        cplx* d = dst.p + line * dst.ls;
#pragma unroll
        for (int p = 0; p < R; ++p) {
            const int e = e0 + p * sub;
            if (e < nvalid) d[e * dst.es] = a[p];
        }
    }
}

// Last forward stage (Ls = R, trivial twiddles) fused with the pointwise multiply by the coefficient spectrum
// and the first inverse stage: the R points never leave registers.  chat: element e of line l at chat[l*cls+e*ces].
template <int R>
__device__ __forceinline__ void mid_stage(Lines src, Lines dst, int nlines, int P, const cplx* __restrict__ chat,
                                          long ces, long cls, int nvalid_in, int nvalid_out) {
    const int nb = P / R;
    const int total = nlines * nb;
    for (int w = threadIdx.x; w < total; w += blockDim.x) {
        const int u = w / nlines, line = w - u * nlines;
        const int e0 = u * R;
        cplx a[R];
        const cplx* s = src.p + line * src.ls;
#pragma unroll
        for (int p = 0; p < R; ++p) a[p] = (e0 + p < nvalid_in) ? s[(e0 + p) * src.es] : make_double2(0.0, 0.0);
        Bfly<R, false>::run(a);
        const cplx* c = chat + line * cls + e0 * ces;
#pragma unroll
        for (int q = 0; q < R; ++q) a[q] = cmul(a[q], __ldg(c + q * ces));
        Bfly<R, true>::run(a);
        cplx* d = dst.p + line * dst.ls;
#pragma unroll
        for (int p = 0; p < R; ++p)
            if (e0 + p < nvalid_out) d[(e0 + p) * dst.es] = a[p];
    }
}

// Runtime-radix dispatch (the radix is uniform over the CTA).
__device__ __forceinline__ void dif_stage_rt(int R, Lines src, Lines dst, int nlines, int P, int Ls, const cplx* tw,
                                             int nvalid) {
    if (R == 8) dif_stage<8>(src, dst, nlines, P, Ls, tw, nvalid);
    else if (R == 4) dif_stage<4>(src, dst, nlines, P, Ls, tw, nvalid);
    else dif_stage<2>(src, dst, nlines, P, Ls, tw, nvalid);
}
__device__ __forceinline__ void dit_stage_rt(int R, Lines src, Lines dst, int nlines, int P, int Ls, const cplx* tw,
                                             int nvalid) {
    if (R == 8) dit_stage<8>(src, dst, nlines, P, Ls, tw, nvalid);
    else if (R == 4) dit_stage<4>(src, dst, nlines, P, Ls, tw, nvalid);
    else dit_stage<2>(src, dst, nlines, P, Ls, tw, nvalid);
}
__device__ __forceinline__ void mid_stage_rt(int R, Lines src, Lines dst, int nlines, int P, const cplx* chat, long ces,
                                             long cls, int nvalid_in, int nvalid_out) {
    if (R == 8) mid_stage<8>(src, dst, nlines, P, chat, ces, cls, nvalid_in, nvalid_out);
    else if (R == 4) mid_stage<4>(src, dst, nlines, P, chat, ces, cls, nvalid_in, nvalid_out);
    else mid_stage<2>(src, dst, nlines, P, chat, ces, cls, nvalid_in, nvalid_out);
}

// Full forward transform of `nlines` lines in place (all stages), CTA-wide; ends with a barrier.
__device__ __forceinline__ void fft_forward(const AxisPlan& ax, Lines v, int nlines, const cplx* tw, int nvalid) {
    int Ls = ax.P;
    for (int s = 0; s < ax.nst; ++s) {
        dif_stage_rt(ax.radix[s], v, v, nlines, ax.P, Ls, tw, s == 0 ? nvalid : ax.P);
        Ls /= ax.radix[s];
        __syncthreads();
    }
}
// Full inverse transform in place; only outputs < nvalid are stored by the last stage; ends with a barrier.
__device__ __forceinline__ void fft_inverse(const AxisPlan& ax, Lines v, int nlines, const cplx* tw, int nvalid) {
    int Ls = 1;
    for (int s = ax.nst - 1; s >= 0; --s) {
        Ls *= ax.radix[s];
        dit_stage_rt(ax.radix[s], v, v, nlines, ax.P, Ls, tw, s == 0 ? nvalid : ax.P);
        __syncthreads();
    }
}

}  // namespace gsm
