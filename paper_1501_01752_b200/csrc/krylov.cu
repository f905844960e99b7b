// krylov.cu - batched lock-step GMRES ("GMRes ... according to Saad with the modified
// Gram-Schmidt orthogonalization"), one instance per (k, omega) point of the scan, all device-resident.
//
// Gram-Schmidt.  Saad's MGS step is  h_i = <v_i, w - sum_{k<i} h_k v_k>, i = 0..j.  Expanding the inner product,
//     h_i = <v_i, w> - sum_{k<i} h_k <v_i, v_k>,
// an identity that needs no orthogonality assumption.  So one streaming sweep over the basis gives every
// <v_i, w> together with the new row <v_i, v_j> of the Gram matrix (sweep_dots), a tiny per-solve recurrence
// gives the same h_i MGS produces up to rounding order (hsolve), and a second streaming sweep forms
// w - sum h_i v_i and its norm (sweep_update).  This replaces the paper's one-CUBLAS-call-per-dot/axpy (5 vector
// passes per basis vector, j grid-wide reductions per iteration) by 2 passes per basis vector and 2 reductions.
// The paper's library calls were made for a GTX Titan; the algebra is kept, the schedule is not.
//
// <u, v> = sum conj(u) v.  Reductions are two-stage and deterministic (per-CTA partials, then a fixed-order sum).
#include "gsm_internal.cuh"
#include "krylov_device.cuh"

namespace gsm {

#define KT 256   // threads per CTA in the sweeps

static __device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

__global__ void krylov_init_kernel(KrylovDims d, KrylovState s, int batch, long i0, long n) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const double* p = s.pol + 6 * b;
    const double beta = sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2] + p[3] * p[3] + p[4] * p[4] + p[5] * p[5]);
    s.beta[b] = beta;
    s.bnorm[b] = beta;
    s.guess[b] = 0;
    s.iters[b] = 0;
    s.active[b] = beta > 0.0 ? 1 : 0;
    if (beta <= 0.0) atomicSub(s.nactive, 1);
    for (int i = 0; i < d.ld; ++i) s.g[(long)b * d.ld + i] = make_double2(0.0, 0.0);
    s.g[(long)b * d.ld] = make_double2(beta, 0.0);
    if (beta > 0.0) {
        cplx* v0 = s.basis + (long)b * d.vlen;
        for (int c = 0; c < 3; ++c) v0[c * n + i0] = make_double2(p[2 * c] / beta, p[2 * c + 1] / beta);
    }
}

// sweep 1: part[b][chunk][2i] = sum_chunk conj(v_i) w, part[..][2i+1] = sum_chunk conj(v_i) v_j, i = 0..j
template <int E>
__global__ void __launch_bounds__(KT) sweep_dots_kernel(KrylovDims d, KrylovState s, int batch, int j) {
    const int b = blockIdx.y;
    if (!s.active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* red = reinterpret_cast<double*>(smem_raw);   // [KT/32][j+1][4]
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
    const long vs = (long)batch * d.vlen;
    const cplx* vb = s.basis + (long)b * d.vlen;
    const cplx* w = vb + (long)(j + 1) * vs;
    const cplx* vj = vb + (long)j * vs;
    cplx wr[E], vr[E];
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        const bool ok = e < d.vlen;
        wr[k] = ok ? w[e] : make_double2(0.0, 0.0);
        vr[k] = ok ? vj[e] : make_double2(0.0, 0.0);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = 0; i <= j; ++i) {
        const cplx* vi = vb + (long)i * vs;
        cplx u[E];
#pragma unroll
        for (int k = 0; k < E; ++k) {
            const long e = e0 + (long)k * KT;
            u[k] = (e < d.vlen) ? vi[e] : make_double2(0.0, 0.0);
        }
        double a0 = 0, a1 = 0, g0 = 0, g1 = 0;
#pragma unroll
        for (int k = 0; k < E; ++k) {   // conj(u) * w, conj(u) * vj
            a0 = fma(u[k].x, wr[k].x, fma(u[k].y, wr[k].y, a0));
            a1 = fma(u[k].x, wr[k].y, fma(-u[k].y, wr[k].x, a1));
            g0 = fma(u[k].x, vr[k].x, fma(u[k].y, vr[k].y, g0));
            g1 = fma(u[k].x, vr[k].y, fma(-u[k].y, vr[k].x, g1));
        }
        a0 = warp_sum(a0); a1 = warp_sum(a1); g0 = warp_sum(g0); g1 = warp_sum(g1);
        if (lane == 0) {
            double* r = red + ((long)warp * (j + 1) + i) * 4;
            r[0] = a0; r[1] = a1; r[2] = g0; r[3] = g1;
        }
    }
    __syncthreads();
    cplx* out = s.part + (long)b * 2 * d.ld * d.nchunk + blockIdx.x;   // part[b][q][chunk]: reductions read contiguously
    for (int i = threadIdx.x; i <= j; i += KT) {
        double a0 = 0, a1 = 0, g0 = 0, g1 = 0;
        for (int wq = 0; wq < KT / 32; ++wq) {
            const double* r = red + ((long)wq * (j + 1) + i) * 4;
            a0 += r[0]; a1 += r[1]; g0 += r[2]; g1 += r[3];
        }
        out[(long)(2 * i) * d.nchunk] = make_double2(a0, a1);
        out[(long)(2 * i + 1) * d.nchunk] = make_double2(g0, g1);
    }
}

// Reduction of sweep 1's partials over the chunks, one CTA per (entry i, solve b): hcol[b][i] = <v_i, w> (before the
// recurrence) and gram[i][j] = <v_i, v_j>.  Threads stride over the chunks, then a fixed shuffle / shared-memory tree:
// deterministic.  (One CTA per solve doing all j + 1 entries took 48 us per iteration at 63^3 orders and 1.4 ms at 256^3,
// profiles/ncu_full_r3_63.txt: a chain of dependent load round trips on one SM.)
#define HS_T 256
__global__ void __launch_bounds__(HS_T) hreduce_kernel(KrylovDims d, KrylovState s, int j) {
    const int i = blockIdx.x, b = blockIdx.y;
    if (!s.active[b]) return;
    __shared__ double red[HS_T / 32][4];
    const cplx* p = s.part + ((long)b * 2 * d.ld + 2 * i) * d.nchunk;
    double a0 = 0, a1 = 0, g0 = 0, g1 = 0;
    for (int c = threadIdx.x; c < d.nchunk; c += HS_T) {
        const cplx a = p[c], g = p[d.nchunk + c];
        a0 += a.x; a1 += a.y; g0 += g.x; g1 += g.y;
    }
    a0 = warp_sum(a0); a1 = warp_sum(a1); g0 = warp_sum(g0); g1 = warp_sum(g1);
    if ((threadIdx.x & 31) == 0) {
        double* r = red[threadIdx.x >> 5];
        r[0] = a0; r[1] = a1; r[2] = g0; r[3] = g1;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        a0 = a1 = g0 = g1 = 0;
        for (int q = 0; q < HS_T / 32; ++q) { a0 += red[q][0]; a1 += red[q][1]; g0 += red[q][2]; g1 += red[q][3]; }
        s.hcol[(long)b * d.ld + i] = make_double2(a0, a1);
        s.gram[(long)b * d.ld * d.ld + (long)i * d.ld + j] = make_double2(g0, g1);
    }
}

// per solve: run the MGS recurrence on the reduced inner products -> hcol[0..j] (warp 0; the others help staging)
__global__ void __launch_bounds__(HS_T) hsolve_kernel(KrylovDims d, KrylovState s, int batch, int j, int stage) {
    const int b = blockIdx.x;
    if (!s.active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* dd = reinterpret_cast<cplx*>(smem_raw);   // [ld]
    cplx* gT = s.gram + (long)b * d.ld * d.ld;      // gT[k*ld + i] = <v_k, v_i>, k <= i
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i <= j; i += HS_T) dd[i] = s.hcol[(long)b * d.ld + i];
    // stage the Gram rows the recurrence needs (k < i <= j) in shared memory: the recurrence is a chain of j dependent
    // steps, and a global-memory load per step would cost an L2 round trip each
    const cplx* gs = gT;                             // stage == 0: basis too long for shared memory, read the rows from global
    if (stage) {
        cplx* gw = dd + d.ld;                        // [j][ld] rows 0..j-1
        for (int q = threadIdx.x; q < j * (j + 1); q += HS_T) {
            const int k = q / (j + 1), i = q - k * (j + 1);
            if (i > k && i < j) gw[k * d.ld + i] = gT[(long)k * d.ld + i];
        }
        __syncthreads();                             // also orders the column-j entries written above
        for (int q = threadIdx.x; q < j; q += HS_T) gw[q * d.ld + j] = gT[(long)q * d.ld + j];
        gs = gw;
    }
    __syncthreads();
    if (warp != 0) return;
    // column-oriented recurrence: once h_k is final, every later d_i loses h_k <v_i, v_k> = h_k conj(<v_k, v_i>)
    for (int k = 0; k < j; ++k) {
        const cplx hk = dd[k];
        for (int i = k + 1 + lane; i <= j; i += 32) {
            const cplx t = cmulc(hk, gs[(long)k * d.ld + i]);
            dd[i] = make_double2(dd[i].x - t.x, dd[i].y - t.y);
        }
        __syncwarp();
    }
    for (int i = lane; i <= j; i += 32) s.hcol[(long)b * d.ld + i] = dd[i];
}

// sweep 2: w <- w - sum_i h_i v_i ; npart[b][chunk] = sum_chunk |w|^2   (stored in part[b][chunk][0].x)
template <int E>
__global__ void __launch_bounds__(KT) sweep_update_kernel(KrylovDims d, KrylovState s, int batch, int j) {
    const int b = blockIdx.y;
    if (!s.active[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* h = reinterpret_cast<cplx*>(smem_raw);   // [j+1]
    __shared__ double wsum[KT / 32];
    for (int i = threadIdx.x; i <= j; i += KT) h[i] = s.hcol[(long)b * d.ld + i];
    __syncthreads();
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
    const long vs = (long)batch * d.vlen;
    const cplx* vb = s.basis + (long)b * d.vlen;
    cplx* w = s.basis + (long)b * d.vlen + (long)(j + 1) * vs;
    cplx wr[E];
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        wr[k] = (e < d.vlen) ? w[e] : make_double2(0.0, 0.0);
    }
    for (int i = 0; i <= j; ++i) {
        const cplx* vi = vb + (long)i * vs;
        const cplx hi = h[i];
#pragma unroll
        for (int k = 0; k < E; ++k) {
            const long e = e0 + (long)k * KT;
            const cplx u = (e < d.vlen) ? vi[e] : make_double2(0.0, 0.0);
            wr[k].x = fma(-hi.x, u.x, fma(hi.y, u.y, wr[k].x));
            wr[k].y = fma(-hi.x, u.y, fma(-hi.y, u.x, wr[k].y));
        }
    }
    double nn = 0.0;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e < d.vlen) {
            w[e] = wr[k];
            nn = fma(wr[k].x, wr[k].x, fma(wr[k].y, wr[k].y, nn));
        }
    }
    nn = warp_sum(nn);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = nn;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < KT / 32; ++q) t += wsum[q];
        s.part[(long)b * 2 * d.ld * d.nchunk + blockIdx.x] = make_double2(t, 0.0);
    }
}

// two-sweep path: h_{j+1,j} = ||w|| from the partial norms of sweep 2, then the Givens step
__global__ void givens_kernel(KrylovDims d, KrylovState s, int batch, int j) {   // one warp per solve
    const int b = blockIdx.x;
    if (!s.active[b]) return;
    double nn = 0.0;
    for (int c = threadIdx.x; c < d.nchunk; c += 32) nn += s.part[(long)b * 2 * d.ld * d.nchunk + c].x;
    nn = warp_sum(nn);
    if (threadIdx.x != 0) return;
    givens_step(d, s, b, j, s.hcol + (long)b * d.ld, sqrt(nn), s.cs + (long)b * d.mmax, s.sn + (long)b * d.mmax);
}

// v_{j+1} = w / h_{j+1,j}
template <int E>
__global__ void __launch_bounds__(KT) normalize_kernel(KrylovDims d, KrylovState s, int batch, int j) {
    const int b = blockIdx.y;
    if (!s.active[b]) return;
    const double sc = s.scale[b];
    cplx* w = s.basis + (long)b * d.vlen + (long)(j + 1) * batch * d.vlen;
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e < d.vlen) {
            const cplx v = w[e];
            w[e] = make_double2(v.x * sc, v.y * sc);
        }
    }
}

// y = R^{-1} g (upper triangular, m = iters[b]).  One warp per solve: the lanes share each row's sum (row i of R is
// contiguous in k), fixed shuffle tree, so the m dependent steps cost one load round trip each instead of m - i.
__global__ void __launch_bounds__(128) backsolve_kernel(KrylovDims d, KrylovState s, int batch, const int* __restrict__ mask) {
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= batch || (mask && !mask[b])) return;
    const int m = s.iters[b];
    const cplx* Rc = s.R + (long)b * d.ld * d.mmax;
    const cplx* g = s.g + (long)b * d.ld;
    cplx* y = s.ycoef + (long)b * d.mmax;
    for (int i = m - 1; i >= 0; --i) {
        cplx acc = make_double2(0.0, 0.0);
        for (int k = i + 1 + lane; k < m; k += 32) acc = cfma(Rc[(long)i * d.mmax + k], y[k], acc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
            acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
        }
        if (lane == 0) {
            const cplx gi = g[i], rii = Rc[(long)i * d.mmax + i];
            const double ax = gi.x - acc.x, ay = gi.y - acc.y;
            const double inv = 1.0 / (rii.x * rii.x + rii.y * rii.y);
            y[i] = make_double2((ax * rii.x + ay * rii.y) * inv, (ay * rii.x - ax * rii.y) * inv);
        }
        __syncwarp();   // y[i] is read by every lane in the next rows
    }
}

// E[b] = x0[b] (if the solve started from a guess) + sum_{i<m} y_i v_i.  x0 may alias out (same thread, same element).
template <int E>
__global__ void __launch_bounds__(KT) combine_kernel(KrylovDims d, KrylovState s, int batch, const cplx* x0, cplx* out,
                                                     const int* __restrict__ mask) {
    const int b = blockIdx.y;
    if (mask && !mask[b]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* y = reinterpret_cast<cplx*>(smem_raw);
    const int m = s.iters[b];
    for (int i = threadIdx.x; i < m; i += KT) y[i] = s.ycoef[(long)b * d.mmax + i];
    __syncthreads();
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
    const long vs = (long)batch * d.vlen;
    const cplx* vb = s.basis + (long)b * d.vlen;
    cplx acc[E];
    const bool g0 = x0 != nullptr && s.guess[b] != 0;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        acc[k] = (g0 && e < d.vlen) ? x0[(long)b * d.vlen + e] : make_double2(0.0, 0.0);
    }
    for (int i = 0; i < m; ++i) {
        const cplx* vi = vb + (long)i * vs;
        const cplx yi = y[i];
#pragma unroll
        for (int k = 0; k < E; ++k) {
            const long e = e0 + (long)k * KT;
            if (e < d.vlen) acc[k] = cfma(yi, vi[e], acc[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e < d.vlen) out[(long)b * d.vlen + e] = acc[k];
    }
}

// partial ||b - y||^2 per chunk, b = pol delta_{m,0}; r_out (may be null) receives b - y
template <int E>
__global__ void __launch_bounds__(KT) resid_part_kernel(KrylovDims d, KrylovState s, int batch, const cplx* __restrict__ y,
                                                        long i0, long n, cplx* __restrict__ r_out) {
    const int b = blockIdx.y;
    if (!r_out && !s.rflag[b]) return;      // final residual of a solve whose guess was accepted: ||r0|| is known
    __shared__ double wsum[KT / 32];
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
    double nn = 0.0;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e < d.vlen) {
            cplx v = y[(long)b * d.vlen + e];
            const long c = e / n, r = e - c * n;
            if (r == i0) { v.x -= s.pol[6 * b + 2 * c]; v.y -= s.pol[6 * b + 2 * c + 1]; }
            if (r_out) r_out[(long)b * d.vlen + e] = make_double2(-v.x, -v.y);
            nn = fma(v.x, v.x, fma(v.y, v.y, nn));
        }
    }
    nn = warp_sum(nn);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = nn;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < KT / 32; ++q) t += wsum[q];
        s.part[(long)b * 2 * d.ld * d.nchunk + blockIdx.x] = make_double2(t, 0.0);
    }
}
__global__ void resid_final_kernel(KrylovDims d, KrylovState s, int batch, double* __restrict__ resid) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    double nn = 0.0;
    for (int c = 0; c < d.nchunk; ++c) nn += s.part[(long)b * 2 * d.ld * d.nchunk + c].x;
    const double r = s.rflag[b] ? sqrt(nn) : s.beta[b];
    resid[b] = s.bnorm[b] > 0.0 ? r / s.bnorm[b] : 0.0;
}
__global__ void residual_select_kernel(KrylovState s, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < batch) s.rflag[b] = (s.guess[b] && s.iters[b] == 0) ? 0 : 1;
}

// initial guess, per solve: beta = ||r0|| from the chunk partials; the guess is taken when it beats the zero start
__global__ void guess_init_kernel(KrylovDims d, KrylovState s, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    double nn = 0.0;
    for (int c = 0; c < d.nchunk; ++c) nn += s.part[(long)b * 2 * d.ld * d.nchunk + c].x;
    const double beta = sqrt(nn), bn = s.bnorm[b];
    if (!(bn > 0.0) || !(beta < bn)) return;      // zero source, or a guess worse than x0 = 0: keep the zero start
    s.guess[b] = 1;
    s.beta[b] = beta;
    s.g[(long)b * d.ld] = make_double2(beta, 0.0);
    if (beta <= s.tol[0] * bn) {                  // the guess already meets the stop test: no iteration
        s.active[b] = 0;
        atomicSub(s.nactive, 1);
    }
}
// v_0 = r0 / beta for the solves that took their guess (r0 sits in basis slot 0 already, unnormalised)
template <int E>
__global__ void __launch_bounds__(KT) guess_v0_kernel(KrylovDims d, KrylovState s, int batch, long i0, long n) {
    const int b = blockIdx.y;
    const bool g = s.guess[b] != 0;
    const double sc = g ? 1.0 / s.beta[b] : 0.0, bn = s.bnorm[b];
    cplx* v0 = s.basis + (long)b * d.vlen;
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e >= d.vlen) continue;
        if (g) {
            const cplx v = v0[e];
            v0[e] = make_double2(v.x * sc, v.y * sc);
        } else {                                  // zero start: v_0 = b / ||b|| (the delta vector of launch_krylov_init)
            const long c = e / n, r = e - c * n;
            v0[e] = (r == i0 && bn > 0.0) ? make_double2(s.pol[6 * b + 2 * c] / bn, s.pol[6 * b + 2 * c + 1] / bn)
                                          : make_double2(0.0, 0.0);
        }
    }
}

// x0[b] = sum_q wgt[b][q] all[nbr[b][q]]  (interpolation of solved neighbours along the mesh, complex weights)
template <int E>
__global__ void __launch_bounds__(KT) mesh_guess_kernel(KrylovDims d, const cplx* __restrict__ all, const int* __restrict__ nbr,
                                                        const cplx* __restrict__ wgt, cplx* __restrict__ x0) {
    const int b = blockIdx.y;
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
    cplx acc[E];
#pragma unroll
    for (int k = 0; k < E; ++k) acc[k] = make_double2(0.0, 0.0);
    for (int q = 0; q < GSM_MESH_NNB; ++q) {
        const int p = nbr[GSM_MESH_NNB * b + q];
        if (p < 0) continue;
        const cplx w = wgt[GSM_MESH_NNB * b + q];
#pragma unroll
        for (int k = 0; k < E; ++k) {
            const long e = e0 + (long)k * KT;
            if (e < d.vlen) acc[k] = cfma(w, all[(long)p * d.vlen + e], acc[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e < d.vlen) x0[(long)b * d.vlen + e] = acc[k];
    }
}
template <int E>
__global__ void __launch_bounds__(KT) mesh_scatter_kernel(KrylovDims d, const cplx* __restrict__ src, const int* __restrict__ idx,
                                                          cplx* __restrict__ all, const int* __restrict__ mask) {
    const int b = blockIdx.y;
    if (mask && !mask[b]) return;
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
    cplx* dst = all + (long)idx[b] * d.vlen;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e < d.vlen) dst[e] = src[(long)b * d.vlen + e];
    }
}

// ---- slot-refill scan (gsm_scan with more points than max_batch; the scan is a list of independent
// solves).  A slot whose solve has finished is given the next pending point at the next tick, so the lock-step batch
// stays full; every solve is at its own Arnoldi index s.iters[b].
// After the Arnoldi step of a tick: fin[b] = 1 if the slot's solve converged in this tick, 2 if it stopped at max_iters;
// rflag[b] (mask of the true-residual apply) = fin[b] != 0.
__global__ void refill_mark_kernel(KrylovDims d, KrylovState s, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    int f = 0;
    if (s.running[b]) {
        if (!s.active[b]) f = 1;
        else if (s.iters[b] >= d.mmax) { s.active[b] = 0; atomicSub(s.nactive, 1); f = 2; }
    }
    s.fin[b] = f;
    s.rflag[b] = f != 0;
}
// One block.  Records the results of the slots that finished (their true residual is in resid_slot, their field in
// E_slot) under their point index, then hands the next pending points to the free slots in slot order (deterministic)
// and initialises their Krylov state as krylov_init_kernel does; newv[b] = 1 where v_0 has to be written.
__global__ void __launch_bounds__(256) refill_commit_kernel(KrylovDims d, KrylovState s, RefillDev r, int batch, long i0, long n,
                                                            const cplx* __restrict__ E_slot, const double* __restrict__ resid_slot,
                                                            double* __restrict__ kvec_slot, double* __restrict__ k0_slot) {
    __shared__ int wcount[8];
    __shared__ int base_sh;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) base_sh = *r.next;
    __syncthreads();
    for (int b0 = 0; b0 < batch; b0 += 256) {
        const int b = b0 + threadIdx.x;
        bool want = false;
        if (b < batch) {
            if (s.fin[b]) {
                const int p = s.point[b];
                r.out_iters[p] = s.iters[b];
                r.out_resid[p] = resid_slot[b];
                for (int c = 0; c < 3; ++c) r.out_resp[3 * (long)p + c] = E_slot[(long)b * d.vlen + c * n + i0];
                r.out_flag[p] = s.fin[b] == 2;
                s.running[b] = 0;
                s.fin[b] = 0;
                atomicAdd(r.ndone, 1);
            }
            want = !s.running[b];
        }
        const unsigned m = __ballot_sync(0xffffffffu, want);
        if (lane == 0) wcount[warp] = __popc(m);
        __syncthreads();
        int before = __popc(m & ((1u << lane) - 1u)), total = 0;
        for (int w = 0; w < 8; ++w) { if (w < warp) before += wcount[w]; total += wcount[w]; }
        const int q = base_sh + before;
        int nv = 0;
        if (want && q < r.npts) {
            s.point[b] = q;
            for (int a = 0; a < 3; ++a) kvec_slot[3 * b + a] = r.kvec_all[3 * (long)q + a];
            k0_slot[b] = r.k0_all[q];
            double* p = s.pol + 6 * b;
            double bb = 0.0;
            for (int a = 0; a < 6; ++a) { p[a] = r.pol_all[6 * (long)q + a]; bb += p[a] * p[a]; }
            const double beta = sqrt(bb);
            s.beta[b] = beta;
            s.bnorm[b] = beta;
            s.guess[b] = 0;
            s.iters[b] = 0;
            s.active[b] = beta > 0.0 ? 1 : 0;
            if (beta > 0.0) atomicAdd(s.nactive, 1);
            for (int i = 0; i < d.ld; ++i) s.g[(long)b * d.ld + i] = make_double2(0.0, 0.0);
            s.g[(long)b * d.ld] = make_double2(beta, 0.0);
            s.running[b] = 1;
            nv = 1;
        }
        if (b < batch) s.newv[b] = nv;
        __syncthreads();
        if (threadIdx.x == 0) base_sh = min(base_sh + total, r.npts);
        __syncthreads();
    }
    if (threadIdx.x == 0) *r.next = base_sh;
}
// v_0 = b / ||b|| (the delta vector at m = 0) for the slots that have just been given a point
template <int E>
__global__ void __launch_bounds__(KT) refill_v0_kernel(KrylovDims d, KrylovState s, int batch, long i0, long n) {
    const int b = blockIdx.y;
    if (!s.newv[b]) return;
    const double bn = s.bnorm[b];
    cplx* v0 = s.basis + (long)b * d.vlen;
    const long e0 = (long)blockIdx.x * (KT * E) + threadIdx.x;
#pragma unroll
    for (int k = 0; k < E; ++k) {
        const long e = e0 + (long)k * KT;
        if (e >= d.vlen) continue;
        const long c = e / n, rr = e - c * n;
        v0[e] = (rr == i0 && bn > 0.0) ? make_double2(s.pol[6 * b + 2 * c] / bn, s.pol[6 * b + 2 * c + 1] / bn)
                                       : make_double2(0.0, 0.0);
    }
}

__global__ void group_count_kernel(KrylovState s, int ngroups, GroupBounds bounds, int* __restrict__ counts) {
    const int g = blockIdx.x;   // one warp per group
    int c = 0;
    for (int b = bounds.b[g] + threadIdx.x; b < bounds.b[g + 1]; b += 32) c += s.active[b] != 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (threadIdx.x == 0) counts[g] = c;
}

// ---- host-side launchers ----------------------------------------------------------------------------------------
#define GSM_E 4   // elements per thread in the sweeps (KrylovDims.chunk = KT * GSM_E)

cudaError_t krylov_init_attributes() {
    cudaError_t e = cudaFuncSetAttribute(sweep_dots_kernel<GSM_E>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hsolve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    return e;
}
cudaError_t launch_krylov_init(const KrylovDims& d, const KrylovState& s, int batch, long i0, long n, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SMALL, st);
    krylov_init_kernel<<<(batch + 127) / 128, 128, 0, st>>>(d, s, batch, i0, n);
    return cudaGetLastError();
}
// The sweeps' algorithmic bytes depend on how many solves are still iterating, which the host does not know at launch
// time: run_batch bills them afterwards from the final iteration counts (sweep_dots (j+2) V: w and v_0..v_j;
// sweep_update (j+3) V: w, v_0..v_j, write w; normalize 2 V).
cudaError_t launch_sweep_dots(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SWEEP_DOTS, st);
    const size_t smem = sizeof(double) * 4 * (KT / 32) * (size_t)(j + 1);
    sweep_dots_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, smem, st>>>(d, s, batch, j);
    return cudaGetLastError();
}
cudaError_t launch_hsolve(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof) {
    { ProfScope pr_(prof, KC_HSOLVE, st);
      hreduce_kernel<<<dim3(j + 1, batch), HS_T, 0, st>>>(d, s, j);
      const cudaError_t e = cudaGetLastError();
      if (e != cudaSuccess) return e; }
    ProfScope ps_(prof, KC_HSOLVE, st);
    size_t smem = sizeof(cplx) * d.ld * (size_t)(j + 1);
    const int stage = smem <= 200 * 1024;
    if (!stage) smem = sizeof(cplx) * d.ld;
    hsolve_kernel<<<batch, HS_T, smem, st>>>(d, s, batch, j, stage);
    return cudaGetLastError();
}
cudaError_t launch_sweep_update(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SWEEP_UPDATE, st);
    sweep_update_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, sizeof(cplx) * (j + 1), st>>>(d, s, batch, j);
    return cudaGetLastError();
}
cudaError_t launch_givens(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_GIVENS, st);
    givens_kernel<<<batch, 32, 0, st>>>(d, s, batch, j);
    return cudaGetLastError();
}
cudaError_t launch_normalize(const KrylovDims& d, const KrylovState& s, int batch, int j, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_NORMALIZE, st);
    normalize_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, s, batch, j);
    return cudaGetLastError();
}
cudaError_t launch_backsolve(const KrylovDims& d, const KrylovState& s, int batch, cudaStream_t st, Profiler* prof,
                             const int* d_mask) {
    ProfScope ps_(prof, KC_SMALL, st);
    backsolve_kernel<<<(batch + 3) / 4, 128, 0, st>>>(d, s, batch, d_mask);
    return cudaGetLastError();
}
cudaError_t launch_krylov_guess(const KrylovDims& d, const KrylovState& s, int batch, long i0, long n, cudaStream_t st,
                                Profiler* prof) {
    const cplx* y = s.basis + (size_t)batch * d.vlen;   // slot 1 holds A x0
    cplx* r0 = s.basis;                                 // slot 0 receives b - A x0, then v_0
    { ProfScope ps_(prof, KC_RESIDUAL, st);
      resid_part_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, s, batch, y, i0, n, r0); }
    { ProfScope ps_(prof, KC_SMALL, st);
      guess_init_kernel<<<(batch + 127) / 128, 128, 0, st>>>(d, s, batch); }
    ProfScope ps_(prof, KC_NORMALIZE, st);
    guess_v0_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, s, batch, i0, n);
    return cudaGetLastError();
}
cudaError_t launch_mesh_guess(const KrylovDims& d, int batch, const cplx* d_all, const int* d_nbr, const cplx* d_wgt,
                              cplx* d_x0, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SMALL, st);
    mesh_guess_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, d_all, d_nbr, d_wgt, d_x0);
    return cudaGetLastError();
}
cudaError_t launch_mesh_scatter(const KrylovDims& d, int batch, const cplx* d_src, const int* d_idx, cplx* d_all,
                                cudaStream_t st, Profiler* prof, const int* d_mask) {
    ProfScope ps_(prof, KC_SMALL, st);
    mesh_scatter_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, d_src, d_idx, d_all, d_mask);
    return cudaGetLastError();
}
cudaError_t launch_combine(const KrylovDims& d, const KrylovState& s, int batch, const cplx* d_x0, cplx* d_E, cudaStream_t st,
                           Profiler* prof, const int* d_mask) {
    ProfScope ps_(prof, KC_COMBINE, st);   // (m_b + 1) V per solve, billed by run_batch from the iteration counts
    combine_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, sizeof(cplx) * d.mmax, st>>>(d, s, batch, d_x0, d_E, d_mask);
    return cudaGetLastError();
}
KrylovState krylov_state_view(const KrylovDims& d, const KrylovState& s, int b0, int* nactive) {
    KrylovState v = s;
    const size_t b = (size_t)b0;
    v.basis = s.basis + b * d.vlen;
    v.part = s.part + b * 2 * d.ld * d.nchunk;
    v.gram = s.gram + b * d.ld * d.ld;
    v.hcol = s.hcol + b * d.ld;
    v.R = s.R + b * d.ld * d.mmax;
    v.cs = s.cs + b * d.mmax;
    v.sn = s.sn + b * d.mmax;
    v.g = s.g + b * d.ld;
    v.ycoef = s.ycoef + b * d.mmax;
    v.hist = s.hist + b * d.mmax;
    v.beta = s.beta + b;
    v.bnorm = s.bnorm + b;
    v.guess = s.guess + b;
    v.rflag = s.rflag + b;
    v.scale = s.scale + b;
    v.active = s.active + b;
    v.iters = s.iters + b;
    v.nactive = nactive;
    v.pol = s.pol + 6 * b;
    v.running = s.running + b;
    v.fin = s.fin + b;
    v.point = s.point + b;
    v.newv = s.newv + b;
    return v;
}
cudaError_t launch_group_count(const KrylovState& s, int ngroups, GroupBounds bounds, int* d_counts, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SMALL, st);
    group_count_kernel<<<ngroups, 32, 0, st>>>(s, ngroups, bounds, d_counts);
    return cudaGetLastError();
}
cudaError_t launch_refill_mark(const KrylovDims& d, const KrylovState& s, int batch, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SMALL, st);
    refill_mark_kernel<<<(batch + 127) / 128, 128, 0, st>>>(d, s, batch);
    return cudaGetLastError();
}
cudaError_t launch_refill_commit(const KrylovDims& d, const KrylovState& s, const RefillDev& r, int batch, long i0, long n,
                                 const cplx* d_E_slot, const double* d_resid_slot, double* d_kvec_slot, double* d_k0_slot,
                                 cudaStream_t st, Profiler* prof) {
    { ProfScope ps_(prof, KC_SMALL, st);
      refill_commit_kernel<<<1, 256, 0, st>>>(d, s, r, batch, i0, n, d_E_slot, d_resid_slot, d_kvec_slot, d_k0_slot); }
    ProfScope ps2_(prof, KC_NORMALIZE, st);
    refill_v0_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, s, batch, i0, n);
    return cudaGetLastError();
}
cudaError_t launch_residual_select(const KrylovDims& d, const KrylovState& s, int batch, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_SMALL, st);
    residual_select_kernel<<<(batch + 127) / 128, 128, 0, st>>>(s, batch);
    return cudaGetLastError();
}
cudaError_t launch_true_residual(const KrylovDims& d, const KrylovState& s, int batch, const cplx* d_y, long i0, long n,
                                 double* d_resid, cudaStream_t st, Profiler* prof) {
    { ProfScope ps_(prof, KC_RESIDUAL, st);
    resid_part_kernel<GSM_E><<<dim3(d.nchunk, batch), KT, 0, st>>>(d, s, batch, d_y, i0, n, nullptr); }
    ProfScope ps2_(prof, KC_SMALL, st);
    resid_final_kernel<<<(batch + 127) / 128, 128, 0, st>>>(d, s, batch, d_resid);
    return cudaGetLastError();
}

}  // namespace gsm
