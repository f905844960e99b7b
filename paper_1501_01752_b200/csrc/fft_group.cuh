// fft_group.cuh - 64-point complex-fp64 transforms by 8-lane groups (see apply64.cu for the scheme): lane u of a group
// runs butterfly u of both radix-8 stages; the 8 x 8 transpose between the stages goes through a warp-private padded
// scratch line.  Used by apply64.cu (pruned: half of the inputs are zero padding / half of the outputs are dropped)
// and apply128.cu (full 64-point transforms as the two branches of a radix-2 split of a pruned 128-point line).
#pragma once
#include "fft_device.cuh"

namespace gsm {

// forward radix-8 with a[4..7] == 0 on entry (zero padding): the first layer of adds disappears
static __device__ __forceinline__ void bfly8_fwd_half_in(cplx* a) {
    // even part from {a0, a2, 0, 0}, odd part from {a1, a3, 0, 0}
    const cplx e0 = cadd(a[0], a[2]), e2 = csub(a[0], a[2]);
    const cplx m2 = mul_mi<false>(a[2]);
    const cplx e1 = cadd(a[0], m2), e3 = csub(a[0], m2);
    const cplx o0 = cadd(a[1], a[3]), o2r = csub(a[1], a[3]);
    const cplx m3 = mul_mi<false>(a[3]);
    const cplx o1r = cadd(a[1], m3), o3r = csub(a[1], m3);
    // o[k] *= w8^k, w8 = exp(-i pi/4)
    const cplx o1 = make_double2((o1r.x + o1r.y) * GSM_SQRT1_2, (o1r.y - o1r.x) * GSM_SQRT1_2);
    const cplx o2 = mul_mi<false>(o2r);
    const cplx o3 = make_double2((o3r.y - o3r.x) * GSM_SQRT1_2, (-o3r.x - o3r.y) * GSM_SQRT1_2);
    a[0] = cadd(e0, o0);  a[4] = csub(e0, o0);
    a[1] = cadd(e1, o1);  a[5] = csub(e1, o1);
    a[2] = cadd(e2, o2);  a[6] = csub(e2, o2);
    a[3] = cadd(e3, o3);  a[7] = csub(e3, o3);
}

// inverse radix-8 producing only outputs 0..3 (the kept half)
static __device__ __forceinline__ void bfly8_inv_half_out(cplx* a) {
    cplx e[4] = {a[0], a[2], a[4], a[6]};
    cplx o[4] = {a[1], a[3], a[5], a[7]};
    Bfly<4, true>::run(e);
    Bfly<4, true>::run(o);
    const cplx o1 = make_double2((o[1].x - o[1].y) * GSM_SQRT1_2, (o[1].y + o[1].x) * GSM_SQRT1_2);
    const cplx o2 = mul_mi<true>(o[2]);
    const cplx o3 = make_double2((-o[3].x - o[3].y) * GSM_SQRT1_2, (o[3].x - o[3].y) * GSM_SQRT1_2);
    a[0] = cadd(e[0], o[0]);
    a[1] = cadd(e[1], o1);
    a[2] = cadd(e[2], o2);
    a[3] = cadd(e[3], o3);
}

#define SC_LINE 72   // padded scratch line: element e lives at e + e/8

// forward 64-point transform of one line held by an 8-lane group.  In: a[0..3] = x[u + 8p] (a[4..7] ignored).
// Out: a[q] = value at position 8u + q.  sc = this line's scratch (SC_LINE complex numbers, warp-private).
static __device__ __forceinline__ void fwd64_group(cplx* a, const cplx* tw, cplx* sc, int u) {
    bfly8_fwd_half_in(a);
    sc[u] = a[0];
#pragma unroll
    for (int q = 1; q < 8; ++q) sc[u + 9 * q] = cmul(a[q], tw[q - 1]);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 8; ++p) a[p] = sc[9 * u + p];
    Bfly<8, false>::run(a);
}

// inverse 64-point transform.  In: a[q] = value at position 8u + q.  Out: a[0..3] = y[u + 8p], p < 4.
static __device__ __forceinline__ void inv64_group(cplx* a, const cplx* tw, cplx* sc, int u) {
    Bfly<8, true>::run(a);
#pragma unroll
    for (int p = 0; p < 8; ++p) sc[9 * u + p] = a[p];
    __syncwarp();
    a[0] = sc[u];
#pragma unroll
    for (int q = 1; q < 8; ++q) a[q] = cmulc(sc[u + 9 * q], tw[q - 1]);
    bfly8_inv_half_out(a);
    __syncwarp();   // the scratch line is free for the next transform
}

static __device__ __forceinline__ void load_group_twiddles(cplx* tw, const cplx* __restrict__ table, int u) {
#pragma unroll
    for (int q = 1; q < 8; ++q) tw[q - 1] = __ldg(table + ((u * q) & 63));
}


// Full variants: all 8 inputs of the first stage live / all 8 outputs of the last inverse stage kept.
static __device__ __forceinline__ void fwd64_group_full(cplx* a, const cplx* tw, cplx* sc, int u) {
    Bfly<8, false>::run(a);
    sc[u] = a[0];
#pragma unroll
    for (int q = 1; q < 8; ++q) sc[u + 9 * q] = cmul(a[q], tw[q - 1]);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < 8; ++p) a[p] = sc[9 * u + p];
    Bfly<8, false>::run(a);
}
static __device__ __forceinline__ void inv64_group_full(cplx* a, const cplx* tw, cplx* sc, int u) {
    Bfly<8, true>::run(a);
#pragma unroll
    for (int p = 0; p < 8; ++p) sc[9 * u + p] = a[p];
    __syncwarp();
    a[0] = sc[u];
#pragma unroll
    for (int q = 1; q < 8; ++q) a[q] = cmulc(sc[u + 9 * q], tw[q - 1]);
    Bfly<8, true>::run(a);
    __syncwarp();   // the scratch line is free for the next transform
}

}  // namespace gsm
