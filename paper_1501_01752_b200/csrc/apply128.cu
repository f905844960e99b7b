// apply128.cu - pass 2 (xy plane convolution) specialised for 128-point x and y axes (33..64 harmonics kept, e.g. the
// 63^3 single solves of BASELINE.json config 5), same W layout as the generic kernel.
//
// A pruned 128-point line (upper half = zero padding) splits by ONE radix-2 decimation-in-frequency step into two full
// 64-point transforms with no additions at all:  even frequencies = FFT64(x[e]),  odd = FFT64(x[e] w128^e),  e < 64.
// The inverse needs only the kept half:  y[e] = IFFT64(even)[e] + conj(w128^e) IFFT64(odd)[e].
// Each 64-point transform is done by an 8-lane group (fft_group.cuh).  Output position of frequency k:
//   pos128(k) = (k & 1) * 64 + ((k >> 1) & 7) * 8 + (k >> 4);  chat128 holds Chat in that order on the x and y axes
// (the z axis keeps the generic network's order, which pass 1 and pass 3 produce and consume).
#include "fft_group.cuh"
#include "gsm_internal.cuh"

namespace gsm {

// A[r][col]: r = y-position (128 rows), 64 columns = x-index i1 rotated by r/8 (conflict-free for both phases).
// chat128[(((pos3 * 128 + r) * 2 + br) * 8 + q) * 8 + u] = Chat at (z-position pos3, x-position br*64 + 8u + q, y-position r).
__global__ void __launch_bounds__(512, 1) xy_conv128_kernel(ApplyGeom g, cplx* __restrict__ W,
                                                            const cplx* __restrict__ chat128,
                                                            const int* __restrict__ active) {
    const int b = blockIdx.z, c = blockIdx.y, pos3 = blockIdx.x;
    if (active && !active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* A = reinterpret_cast<cplx*>(smem_raw);   // [128][64]
    cplx* scratch = A + 128 * 64;                  // [64 lines][SC_LINE]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, u = lane & 7, ln = lane >> 3;
    const int N1 = g.N1, N2 = g.N2;
    const cplx* __restrict__ w128 = g.tw[0];       // exp(-2 pi i k / 128)
    cplx tw[7];                                    // w64^(u q) = w128^(2 u q)
#pragma unroll
    for (int q = 1; q < 8; ++q) tw[q - 1] = __ldg(w128 + ((2 * u * q) & 127));
    cplx* sc = scratch + (warp * 4 + ln) * SC_LINE;
    cplx* Wp = W + (((long)b * 3 + c) * g.ax[2].P + pos3) * g.NL;
    cplx a[8], a1[8];

    {   // ---- y forward: 64 groups = 64 lines i1
        const int i1 = warp * 4 + ln;
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int i2 = u + 8 * p;
            a[p] = (i1 < N1 && i2 < N2) ? Wp[i1 * N2 + i2] : make_double2(0.0, 0.0);
            a1[p] = cmul(a[p], __ldg(w128 + i2));
        }
        fwd64_group_full(a, tw, sc, u);
#pragma unroll
        for (int q = 0; q < 8; ++q) A[(8 * u + q) * 64 + ((i1 + u) & 63)] = a[q];
        fwd64_group_full(a1, tw, sc, u);
#pragma unroll
        for (int q = 0; q < 8; ++q) A[(64 + 8 * u + q) * 64 + ((i1 + 8 + u) & 63)] = a1[q];
    }
    __syncthreads();
    // ---- x: per row r, forward (two branches), * Chat, inverse, recombine the kept half, in place
#pragma unroll 1
    for (int round = 0; round < 2; ++round) {
        const int r = round * 64 + warp * 4 + ln;
        cplx* Ar = A + r * 64;
        const int rot = r >> 3;
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int i1 = u + 8 * p;
            a[p] = (i1 < N1) ? Ar[(i1 + rot) & 63] : make_double2(0.0, 0.0);
            a1[p] = cmul(a[p], __ldg(w128 + i1));
        }
        const cplx* cp = chat128 + ((long)(pos3 * 128 + r) * 128) + u;
        fwd64_group_full(a, tw, sc, u);
#pragma unroll
        for (int q = 0; q < 8; ++q) a[q] = cmul(a[q], __ldg(cp + 8 * q));
        inv64_group_full(a, tw, sc, u);
        fwd64_group_full(a1, tw, sc, u);
#pragma unroll
        for (int q = 0; q < 8; ++q) a1[q] = cmul(a1[q], __ldg(cp + 64 + 8 * q));
        inv64_group_full(a1, tw, sc, u);
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int i1 = u + 8 * p;
            const cplx t = cmulc(a1[p], __ldg(w128 + i1));
            if (i1 < N1) Ar[(i1 + rot) & 63] = cadd(a[p], t);
        }
    }
    __syncthreads();
    {   // ---- y inverse
        const int i1 = warp * 4 + ln;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            a[q] = A[(8 * u + q) * 64 + ((i1 + u) & 63)];
            a1[q] = A[(64 + 8 * u + q) * 64 + ((i1 + 8 + u) & 63)];
        }
        inv64_group_full(a, tw, sc, u);
        inv64_group_full(a1, tw, sc, u);
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            const int i2 = u + 8 * p;
            const cplx t = cmulc(a1[p], __ldg(w128 + i2));
            if (i1 < N1 && i2 < N2) Wp[i1 * N2 + i2] = cadd(a[p], t);
        }
    }
}

// chat128 from the generic Chat [P3][128][128] (generic position order on every axis): gen1[p], gen2[p] give the
// generic position of the frequency that sits at new position p on the x resp. y axis.
__global__ void chat128_layout_kernel(const cplx* __restrict__ chat, int P3, const int* __restrict__ gen1,
                                      const int* __restrict__ gen2, cplx* __restrict__ chat128) {
    const long total = (long)P3 * 128 * 128;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int u = (int)(i & 7), q = (int)((i >> 3) & 7), br = (int)((i >> 6) & 1), r = (int)((i >> 7) & 127);
        const long p3 = i >> 14;
        const int p1 = br * 64 + 8 * u + q;
        chat128[i] = chat[(p3 * 128 + gen1[p1]) * 128 + gen2[r]];
    }
}

static const size_t XY128_SMEM = sizeof(cplx) * (128 * 64 + 64 * SC_LINE);

bool apply128_usable(const ApplyGeom& g) {
    return g.ax[0].P == 128 && g.ax[1].P == 128 && g.N1 <= 64 && g.N2 <= 64;
}
// frequency at position p of the radix-2 x (8 x 8) network
int apply128_freq_of_pos(int p) { return (p >> 6) + 2 * (((p >> 3) & 7) + 8 * (p & 7)); }

cudaError_t launch_chat128_layout(const cplx* d_chat, int P3, const int* d_gen1, const int* d_gen2, cplx* d_chat128,
                                  cudaStream_t st) {
    chat128_layout_kernel<<<1024, 256, 0, st>>>(d_chat, P3, d_gen1, d_gen2, d_chat128);
    return cudaGetLastError();
}
cudaError_t launch_xy_conv128(const ApplyGeom& g, int batch, cplx* d_W, const cplx* d_chat128, const int* d_active,
                              cudaStream_t st) {
    xy_conv128_kernel<<<dim3(g.ax[2].P, 3, batch), 512, XY128_SMEM, st>>>(g, d_W, d_chat128, d_active);
    return cudaGetLastError();
}
cudaError_t apply128_init_attributes() {
    return cudaFuncSetAttribute(xy_conv128_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)XY128_SMEM);
}

}  // namespace gsm
