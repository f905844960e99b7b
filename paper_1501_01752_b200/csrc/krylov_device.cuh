// krylov_device.cuh - device code shared by the two Arnoldi variants (krylov.cu two-sweep, arnoldi_cluster.cu MGS).
#pragma once
#include "gsm_internal.cuh"

namespace gsm {

// Givens least squares for one solve (Saad Alg. 6.9 / 6.5.3): rotate the new Hessenberg column h[0..j] (with
// h_{j+1,j} = hn) by the previous rotations, form the new one, update g, record the residual estimate and the stop
// test (readings R9, R23).  h, cs_prev, sn_prev may live in shared or global memory.
__device__ __forceinline__ void givens_step(const KrylovDims& d, const KrylovState& s, int b, int j, const cplx* h, double hn,
                                   const double* cs_prev, const cplx* sn_prev) {
    cplx* Rc = s.R + (long)b * d.ld * d.mmax;     // Rc[i * mmax + j]
    double* cs = s.cs + (long)b * d.mmax;
    cplx* sn = s.sn + (long)b * d.mmax;
    cplx* g = s.g + (long)b * d.ld;
    cplx hi = h[0];
    double col2 = hi.x * hi.x + hi.y * hi.y + hn * hn;   // ||(h_0j .. h_jj, h_{j+1,j})||^2 = ||A v_j||^2 up to rounding
    for (int i = 0; i < j; ++i) {   // previous rotations on the new column
        const cplx hn1 = h[i + 1];
        col2 += hn1.x * hn1.x + hn1.y * hn1.y;
        const double ci = cs_prev[i];
        const cplx si = sn_prev[i];
        const cplx t = cadd(make_double2(ci * hi.x, ci * hi.y), cmul(si, hn1));
        const cplx u = csub(make_double2(ci * hn1.x, ci * hn1.y), cmulc(hi, si));   // -conj(sn) hi + cs hn1
        Rc[(long)i * d.mmax + j] = t;
        hi = u;
    }
    const cplx a = hi;
    const double aa = hypot(a.x, a.y);
    const double r = hypot(aa, hn);
    double c;
    cplx sv;
    if (r == 0.0) { c = 1.0; sv = make_double2(0.0, 0.0); }
    else if (aa == 0.0) { c = 0.0; sv = make_double2(1.0, 0.0); }
    else { c = aa / r; sv = make_double2(a.x / aa * hn / r, a.y / aa * hn / r); }   // (a/|a|) conj(hn)/r, hn real
    cs[j] = c;
    sn[j] = sv;
    Rc[(long)j * d.mmax + j] = cadd(make_double2(c * a.x, c * a.y), make_double2(sv.x * hn, sv.y * hn));
    const cplx gj = g[j];
    const cplx gn = make_double2(-(sv.x * gj.x + sv.y * gj.y), -(sv.x * gj.y - sv.y * gj.x));   // -conj(sn) g_j
    g[j + 1] = gn;
    g[j] = make_double2(c * gj.x, c * gj.y);
    const double res = hypot(gn.x, gn.y) / s.bnorm[b];
    s.hist[(long)b * d.mmax + j] = res;
    s.iters[b] = j + 1;
    // reading R23: the new direction has vanished relative to the vector it was orthogonalised from.  Scale-free, so a
    // solve started from a guess (||r0|| tiny against ||b||) is guarded exactly like a zero start.
    const bool lucky = hn <= 2.220446049250313e-16 * sqrt(col2);
    if (res <= s.tol[0] || lucky) {
        s.active[b] = 0;
        atomicSub(s.nactive, 1);
    } else {
        s.scale[b] = 1.0 / hn;
    }
}

}  // namespace gsm
