// plan_kernels.cu - plan-time device work: the permittivity harmonics c_d = (Delta eps/eps_b)_d
// from analytic Fourier images or from an FFT of a voxel grid, and their circulant spectrum.
#include "gsm_internal.cuh"

namespace gsm {

// 3 (sin x - x cos x) / x^3 : Fourier image of the unit ball (textbook; reading R5)
static __device__ double ball_form(double x) {
    const double x2 = x * x;
    if (x2 < 0.25) {   // series sum_k (-1)^k 3 (2k+2) / (2k+3)! x^(2k); avoids the cancellation at small x
        double term = 1.0, sum = 1.0;
        for (int k = 1; k <= 10; ++k) {
            term *= -x2 / ((double)(2 * k) * (double)(2 * k + 3));   // ratio of consecutive coefficients
            sum += term;
        }
        return sum;
    }
    double s, c;
    sincos(x, &s, &c);
    return 3.0 * (s - x * c) / (x2 * x);
}
static __device__ double sinc_form(double t) { return fabs(t) < 1e-300 ? 1.0 : sin(t) / t; }

// int_P exp(-i G.r) d^3r of a polyhedron, divergence theorem twice:
//   (i / |G|^2) sum_faces (G.n) I_f,  I_f = (i / |G_t|^2) sum_edges (G_t.m) L exp(-i G.mid) sinc(G.half)  or, for G normal
//   to the face (G_t = 0), I_f = area exp(-i G.p0).  G = 0: the volume.
static __device__ cplx polyhedron_image(const ShapeDev& q, const PolyFace* __restrict__ faces,
                                        const PolyEdge* __restrict__ edges, double G1, double G2, double G3) {
    const double g2 = G1 * G1 + G2 * G2 + G3 * G3;
    if (g2 == 0.0) return make_double2(q.vol, 0.0);
    double sr = 0.0, si = 0.0;
    for (int f = q.f0; f < q.f0 + q.nf; ++f) {
        const PolyFace F = faces[f];
        const double Gn = G1 * F.n[0] + G2 * F.n[1] + G3 * F.n[2];
        const double t1 = G1 - Gn * F.n[0], t2 = G2 - Gn * F.n[1], t3 = G3 - Gn * F.n[2];
        const double gt2 = t1 * t1 + t2 * t2 + t3 * t3;
        double ir, ii;
        if (gt2 < 1e-18 * g2) {
            double s, c;
            sincos(-(G1 * F.p0[0] + G2 * F.p0[1] + G3 * F.p0[2]), &s, &c);
            ir = F.area * c; ii = F.area * s;
        } else {
            double ar = 0.0, ai = 0.0;
            for (int e = F.e0; e < F.e0 + F.ne; ++e) {
                const PolyEdge E = edges[e];
                const double x = G1 * E.half[0] + G2 * E.half[1] + G3 * E.half[2];
                const double w = (t1 * E.mL[0] + t2 * E.mL[1] + t3 * E.mL[2]) * (fabs(x) < 1e-8 ? 1.0 - x * x / 6.0 : sin(x) / x);
                double s, c;
                sincos(-(G1 * E.mid[0] + G2 * E.mid[1] + G3 * E.mid[2]), &s, &c);
                ar += w * c; ai += w * s;
            }
            ir = -ai / gt2; ii = ar / gt2;      // times i / |G_t|^2
        }
        sr += Gn * ir; si += Gn * ii;
    }
    return make_double2(-si / g2, sr / g2);     // times i / |G|^2
}

__global__ void coeffs_analytic_kernel(const ShapeDev* __restrict__ sh, int nsh, const PolyFace* __restrict__ faces,
                                       const PolyEdge* __restrict__ edges, double c0r, double c0i, double K1,
                                       double K2, double K3, int N1, int N2, int N3, cplx* __restrict__ coef) {
    const int D1 = 2 * N1 - 1, D2 = 2 * N2 - 1, D3 = 2 * N3 - 1;
    const long total = (long)D1 * D2 * D3;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int j3 = (int)(i % D3), j2 = (int)((i / D3) % D2), j1 = (int)(i / ((long)D3 * D2));
        const double G1 = (j1 - (N1 - 1)) * K1, G2 = (j2 - (N2 - 1)) * K2, G3 = (j3 - (N3 - 1)) * K3;
        double re = 0.0, im = 0.0;
        if (j1 == N1 - 1 && j2 == N2 - 1 && j3 == N3 - 1) { re = c0r; im = c0i; }
        for (int s = 0; s < nsh; ++s) {
            const ShapeDev q = sh[s];
            double S, Si = 0.0;
            if (q.kind == GSM_SPHERE) S = ball_form(sqrt(G1 * G1 + G2 * G2 + G3 * G3) * q.s[0]);
            else if (q.kind == GSM_ELLIPSOID) {
                const double a = G1 * q.s[0], b = G2 * q.s[1], c = G3 * q.s[2];
                S = ball_form(sqrt(a * a + b * b + c * c));
            } else if (q.kind == GSM_POLYHEDRON) {
                const cplx F = polyhedron_image(q, faces, edges, G1, G2, G3);
                S = F.x; Si = F.y;
            } else S = sinc_form(0.5 * G1 * q.s[0]) * sinc_form(0.5 * G2 * q.s[1]) * sinc_form(0.5 * G3 * q.s[2]);
            double ps, pc;
            sincos(-(G1 * q.c[0] + G2 * q.c[1] + G3 * q.c[2]), &ps, &pc);
            // (dre + i dim) * f (S + i Si) * (pc + i ps)
            const double wr = q.f * (S * pc - Si * ps), wi = q.f * (S * ps + Si * pc);
            re += q.dre * wr - q.dim * wi;
            im += q.dre * wi + q.dim * wr;
        }
        coef[i] = make_double2(re, im);
    }
}

cudaError_t launch_coeffs_analytic(const ShapeDev* d_shapes, int nshapes, const PolyFace* d_faces, const PolyEdge* d_edges,
                                   double c0_re, double c0_im, const double K[3], const int N[3], cplx* d_coef,
                                   cudaStream_t st) {
    const long total = (long)(2 * N[0] - 1) * (2 * N[1] - 1) * (2 * N[2] - 1);
    const int grid = (int)((total + 255) / 256 < 4096 ? (total + 255) / 256 : 4096);
    coeffs_analytic_kernel<<<grid, 256, 0, st>>>(d_shapes, nshapes, d_faces, d_edges, c0_re, c0_im, K[0], K[1], K[2], N[0],
                                                 N[1], N[2], d_coef);
    return cudaGetLastError();
}

// c_d -> pad[(d1 mod P1)][(d2 mod P2)][(d3 mod P3)], zero elsewhere (circulant embedding, reading R2)
__global__ void embed_kernel(const cplx* __restrict__ coef, int N1, int N2, int N3, int P1, int P2, int P3,
                             cplx* __restrict__ pad) {
    const int D1 = 2 * N1 - 1, D2 = 2 * N2 - 1, D3 = 2 * N3 - 1;
    const long total = (long)D1 * D2 * D3;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int j3 = (int)(i % D3), j2 = (int)((i / D3) % D2), j1 = (int)(i / ((long)D3 * D2));
        const int p1 = (j1 - (N1 - 1) + P1) % P1, p2 = (j2 - (N2 - 1) + P2) % P2, p3 = (j3 - (N3 - 1) + P3) % P3;
        pad[((long)p1 * P2 + p2) * P3 + p3] = coef[i];
    }
}
cudaError_t launch_embed(const cplx* d_coef, const int N[3], const int P[3], cplx* d_pad, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(d_pad, 0, sizeof(cplx) * (size_t)P[0] * P[1] * P[2], st);
    if (e != cudaSuccess) return e;
    embed_kernel<<<1024, 256, 0, st>>>(d_coef, N[0], N[1], N[2], P[0], P[1], P[2], d_pad);
    return cudaGetLastError();
}

// Forward transform along the middle axis of a dense [outer][P][inner] array, TL lines per CTA, same network as
// the hot path (so the result is in the same position order).
#define GSM_PLAN_TL 8
__global__ void __launch_bounds__(256) fft_axis_kernel(cplx* __restrict__ data, long nlines, AxisPlan ax, long inner,
                                                       const cplx* __restrict__ twg) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);
    cplx* S = tw + ax.P;   // S[e * (TL+1) + line]
    const int P = ax.P, st = GSM_PLAN_TL + 1;
    const long lid0 = (long)blockIdx.x * GSM_PLAN_TL;
    const int nl = (int)min((long)GSM_PLAN_TL, nlines - lid0);
    for (int i = threadIdx.x; i < P; i += blockDim.x) tw[i] = twg[i];
    for (int i = threadIdx.x; i < nl * P; i += blockDim.x) {
        int e, l;
        if (inner == 1) { l = i / P; e = i - l * P; } else { e = i / nl; l = i - e * nl; }
        const long lid = lid0 + l;
        S[e * st + l] = data[(lid / inner) * P * inner + (long)e * inner + lid % inner];
    }
    __syncthreads();
    fft_forward(ax, Lines{S, st, 1}, nl, tw, P);
    for (int i = threadIdx.x; i < nl * P; i += blockDim.x) {
        int e, l;
        if (inner == 1) { l = i / P; e = i - l * P; } else { e = i / nl; l = i - e * nl; }
        const long lid = lid0 + l;
        data[(lid / inner) * P * inner + (long)e * inner + lid % inner] = S[e * st + l];
    }
}
cudaError_t launch_fft_axis(cplx* d_data, long outer, const AxisPlan& ax, long inner, const cplx* d_tw, cudaStream_t st) {
    if (ax.P == 1) return cudaSuccess;
    const long nlines = outer * inner;
    const size_t smem = sizeof(cplx) * ((size_t)ax.P + (size_t)ax.P * (GSM_PLAN_TL + 1));
    fft_axis_kernel<<<(unsigned)((nlines + GSM_PLAN_TL - 1) / GSM_PLAN_TL), 256, smem, st>>>(d_data, nlines, ax, inner, d_tw);
    return cudaGetLastError();
}

// chat[pos3][pos1][pos2] = padfft[pos1][pos2][pos3] / (P1 P2 P3)   (inverse-transform scaling folded in here)
__global__ void chat_layout_kernel(const cplx* __restrict__ in, int P1, int P2, int P3, cplx* __restrict__ out) {
    const long total = (long)P1 * P2 * P3;
    const double sc = 1.0 / (double)total;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int p2 = (int)(i % P2), p1 = (int)((i / P2) % P1), p3 = (int)(i / ((long)P2 * P1));
        const cplx v = in[((long)p1 * P2 + p2) * P3 + p3];
        out[i] = make_double2(v.x * sc, v.y * sc);
    }
}
cudaError_t launch_chat_layout(const cplx* d_padfft, const int P[3], cplx* d_chat, cudaStream_t st) {
    chat_layout_kernel<<<1024, 256, 0, st>>>(d_padfft, P[0], P[1], P[2], d_chat);
    return cudaGetLastError();
}

// voxel path: g_j = (eps_j - eps_b) / eps_b (Eq. 4) or 1 - eps_b / eps_j (Eq. 5) in place
__global__ void voxel_prepare_kernel(cplx* __restrict__ grid, long count, double br, double bi, int hform) {
    const double inv = 1.0 / (br * br + bi * bi);
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < count; i += (long)gridDim.x * blockDim.x) {
        const cplx e = grid[i];
        if (hform) {   // 1 - eps_b / eps = (eps - eps_b) / eps
            const double nr = e.x - br, ni = e.y - bi, ie = 1.0 / (e.x * e.x + e.y * e.y);
            grid[i] = make_double2((nr * e.x + ni * e.y) * ie, (ni * e.x - nr * e.y) * ie);
            continue;
        }
        const double nr = e.x - br, ni = e.y - bi;
        grid[i] = make_double2((nr * br + ni * bi) * inv, (ni * br - nr * bi) * inv);
    }
}
cudaError_t launch_voxel_prepare(cplx* d_grid, long count, double epsb_re, double epsb_im, int hform, cudaStream_t st) {
    voxel_prepare_kernel<<<1024, 256, 0, st>>>(d_grid, count, epsb_re, epsb_im, hform);
    return cudaGetLastError();
}

// c_d = FFT(g)[pos(d mod Nv)] / (Nv1 Nv2 Nv3); posA[f] = position of frequency f after the forward network
__global__ void voxel_extract_kernel(const cplx* __restrict__ gf, int V1, int V2, int V3, int N1, int N2, int N3,
                                     const int* __restrict__ pos1, const int* __restrict__ pos2,
                                     const int* __restrict__ pos3, cplx* __restrict__ coef) {
    const int D1 = 2 * N1 - 1, D2 = 2 * N2 - 1, D3 = 2 * N3 - 1;
    const long total = (long)D1 * D2 * D3;
    const double sc = 1.0 / ((double)V1 * V2 * V3);
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int j3 = (int)(i % D3), j2 = (int)((i / D3) % D2), j1 = (int)(i / ((long)D3 * D2));
        const int f1 = (j1 - (N1 - 1) + V1) % V1, f2 = (j2 - (N2 - 1) + V2) % V2, f3 = (j3 - (N3 - 1) + V3) % V3;
        const cplx v = gf[((long)pos1[f1] * V2 + pos2[f2]) * V3 + pos3[f3]];
        coef[i] = make_double2(v.x * sc, v.y * sc);
    }
}
cudaError_t launch_voxel_extract(const cplx* d_gridfft, const int Nv[3], const int N[3], const int* d_pos1,
                                 const int* d_pos2, const int* d_pos3, cplx* d_coef, cudaStream_t st) {
    voxel_extract_kernel<<<1024, 256, 0, st>>>(d_gridfft, Nv[0], Nv[1], Nv[2], N[0], N[1], N[2], d_pos1, d_pos2, d_pos3,
                                               d_coef);
    return cudaGetLastError();
}

// Voxel grids whose sizes are not powers of two: the harmonics |d| <= N - 1 of one axis by the defining sum
//   out[o][j][i] = (1 / V) sum_k in[o][k][i] exp(-2 pi i d k / V),  d = j - (N - 1),
// with the phase index (d k) mod V taken in integers and the twiddle from sincospi (exact argument reduction).
__global__ void __launch_bounds__(256) voxel_dft_axis_kernel(const cplx* __restrict__ in, long outer, int V, long inner,
                                                             int N, cplx* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* tw = reinterpret_cast<cplx*>(smem_raw);   // exp(-2 pi i q / V), q = 0..V-1
    for (int q = threadIdx.x; q < V; q += blockDim.x) {
        double s, c;
        sincospi(-2.0 * (double)q / (double)V, &s, &c);
        tw[q] = make_double2(c, s);
    }
    __syncthreads();
    const int D = 2 * N - 1;
    const long total = outer * D * inner;
    const double sc = 1.0 / (double)V;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const long ii = i % inner, j = (i / inner) % D, o = i / (inner * D);
        const long d = ((j - (N - 1)) % V + V) % V;
        const cplx* src = in + o * V * inner + ii;
        cplx acc = make_double2(0.0, 0.0);
        long q = 0;
        for (int k = 0; k < V; ++k) {
            acc = cfma(src[(long)k * inner], tw[q], acc);
            q += d;
            if (q >= V) q -= V;
        }
        out[i] = make_double2(acc.x * sc, acc.y * sc);
    }
}
cudaError_t launch_voxel_dft_axis(const cplx* d_in, long outer, int V, long inner, int N, cplx* d_out, cudaStream_t st) {
    const long total = outer * (2 * N - 1) * inner;
    const int grid = (int)((total + 255) / 256 < 8192 ? (total + 255) / 256 : 8192);
    voxel_dft_axis_kernel<<<grid, 256, sizeof(cplx) * (size_t)V, st>>>(d_in, outer, V, inner, N, d_out);
    return cudaGetLastError();
}

}  // namespace gsm

namespace gsm {
cudaError_t plan_init_attributes() {
    return cudaFuncSetAttribute(fft_axis_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
}
}  // namespace gsm
