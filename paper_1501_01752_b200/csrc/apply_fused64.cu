// apply_fused64.cu - the whole operator apply y = x - G (T x) of Eq. 4 for 64-point axes
// (17..32 harmonics kept per axis, e.g. the 31^3 configs of BASELINE.json) in ONE persistent launch, with the
// z-transformed intermediate W kept in L2 instead of HBM.
//
// The three passes of apply.cu (z forward -> xy plane convolution -> z inverse + Green dyadic) become three kinds of
// work items handed out by an in-order ticket counter to persistent CTAs (2 per SM):
//   Z1(p, tile)  z-FFT of 32 z-lines of solve p, all three components      x            -> Wring[p % RING]
//   XY(p, pos3)  plane convolution of the three component planes at pos3   Wring        -> Wring (in place)
//   Z3(p, tile)  inverse z-FFT of 32 z-lines + Green dyadic                Wring, x     -> y
// Tickets are ordered in slots: slot s holds Z1(s), XY(s - LAG2), Z3(s - LAG3), interleaved so that the HBM-bound Z
// items and the shared-memory/fp64-bound XY items run on the same SM at the same time.  Dependencies are per-solve
// completion counters in global memory (release: barrier + fence + atomicAdd; acquire: ld.acquire spin by one thread +
// barrier).  An item only ever waits for items with SMALLER ticket numbers, and a CTA takes tickets in increasing
// order, so the oldest unfinished ticket is always running and never waits: no deadlock, whatever the number of
// resident CTAs.  W lives in a ring of RING solve slots (RING * 2.06 V, 47 MB at 31^3): a slot is rewritten while its
// lines are still in L2, so W never travels to HBM; the HBM traffic of an apply is x once and y once.
// W is read with L1-bypassing loads (ld.global.cg / cp.async.cg): ring slots are rewritten within one launch.
#include "fft_group.cuh"
#include "gsm_internal.cuh"

namespace gsm {

#ifndef F64_RING
#define F64_RING 16
#define F64_LAG2 3
#define F64_LAG3 6
#endif
#define F64_T 256

static __device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// wait until *p >= need (one thread polls with relaxed loads - an acquire load per poll would invalidate the SM's L1
// every time - and fences once the count is there), then release the CTA
static __device__ __forceinline__ void wait_count(const int* p, int need) {
    if (threadIdx.x == 0) {
        while (ld_relaxed_gpu(p) < need) __nanosleep(256);
        __threadfence();
    }
    __syncthreads();
}
// all global writes of this CTA's item become visible before the counter moves
static __device__ __forceinline__ void signal_count(int* p) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(p, 1);
    }
}

static __device__ __forceinline__ void cp_async16_cg(void* dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
static __device__ __forceinline__ void cp_async_commit_() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> static __device__ __forceinline__ void cp_async_wait_() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct Lane64 {
    int lane, warp, u, ln;
};

// ---- Z1: forward z-FFT of 32 lines x 3 components -----------------------------------------------------------------
// Each 8-lane group loads its line's <= 32 inputs straight from x, transforms (upper half = zero padding, never
// loaded), drops the 64 outputs into a [pos3][32 lines] tile (columns rotated by pos3/8: conflict-free), which goes out
// to W[c][pos3][l] as 512-byte rows.  H-form (Eq. 5): the transform acts on (k x x).
template <bool HFORM>
static __device__ __forceinline__ void z1_item(const ApplyGeom& g, const cplx* __restrict__ xb, cplx* Ws,
                                               const double* __restrict__ kv, int tile, cplx* T, cplx* sc,
                                               const cplx* tw, const Lane64& L) {
    const int N3 = g.N3, NL = g.NL, u = L.u;
    const int l0 = tile * 32, line = L.warp * 4 + L.ln, l = l0 + line;
    const int col = (line + u) & 31;
    const bool lv = l < NL;
    double kk[3];
    if (HFORM) {
        const int i1 = l / g.N2, i2 = l - i1 * g.N2;
        kk[0] = kv[0] + (i1 + g.mmin[0]) * g.K[0];
        kk[1] = kv[1] + (i2 + g.mmin[1]) * g.K[1];
        kk[2] = kv[2] + g.mmin[2] * g.K[2];
    }
    auto load = [&](cplx* a, int c) {
        if (!HFORM) {
            const cplx* xs = xb + (long)c * g.n + (long)l * N3;
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int i3 = u + 8 * p;
                a[p] = (lv && i3 < N3) ? xs[i3] : make_double2(0.0, 0.0);
            }
        } else {   // (k x x)_c = k_c1 x_c2 - k_c2 x_c1
            const int c1 = c == 2 ? 0 : c + 1, c2 = c1 == 2 ? 0 : c1 + 1;
            const cplx* x1 = xb + (long)c1 * g.n + (long)l * N3;
            const cplx* x2 = xb + (long)c2 * g.n + (long)l * N3;
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int i3 = u + 8 * p;
                if (lv && i3 < N3) {
                    const double ka = c1 == 2 ? kk[2] + i3 * g.K[2] : kk[c1], kb = c2 == 2 ? kk[2] + i3 * g.K[2] : kk[c2];
                    const cplx v1 = x1[i3], v2 = x2[i3];
                    a[p] = make_double2(ka * v2.x - kb * v1.x, ka * v2.y - kb * v1.y);
                } else {
                    a[p] = make_double2(0.0, 0.0);
                }
            }
        }
    };
    cplx a[8], nx[4];
    load(nx, 0);
#pragma unroll 1
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int p = 0; p < 4; ++p) a[p] = nx[p];
        if (c < 2) load(nx, c + 1);
        fwd64_group(a, tw, sc, u);
#pragma unroll
        for (int q = 0; q < 8; ++q) T[(8 * u + q) * 32 + col] = a[q];
        __syncthreads();
        cplx* Wd = Ws + (long)c * 64 * NL + l0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int r = k * 8 + L.warp;                  // one 512-byte row per warp and step
            const int ll = (L.lane - (r >> 3)) & 31;       // logical line stored in physical column `lane`
            if (l0 + ll < NL) Wd[(long)r * NL + ll] = T[r * 32 + L.lane];
        }
        __syncthreads();                                   // the tile is rewritten by the next component
    }
}

// ---- XY: plane convolution at one z-position, the three components in turn ------------------------------------------
// A[r][col]: row r = y-position (64), 32 columns = x-index i1 rotated by r/8 (conflict-free in both phases).
//   y forward : group (i1 = 4 warp + ln) reads its 4 x 8 inputs from W (contiguous in i2), writes rows of A
//   x         : group (row r) reads <= 32 inputs from A, forward, * Chat, inverse, writes the kept 32 back in place
//   y inverse : mirror of y forward, stores to W
// chat64[((pos3 * 64 + r) * 8 + q) * 8 + u] = Chat[pos3][pos1 = 8u + q][pos2 = r].
static __device__ __forceinline__ void xy_item(const ApplyGeom& g, cplx* Ws, int pos3, const cplx* __restrict__ chat64,
                                               cplx* A, cplx* sc, const cplx* tw, const Lane64& L) {
    const int N1 = g.N1, N2 = g.N2, u = L.u;
    const long cstride = 64L * g.NL;
    cplx* Wp = Ws + (long)pos3 * g.NL;              // component 0; component c at + c * cstride
    const int i1y = L.warp * 4 + L.ln;              // y-phase line of this group
    cplx a[8], nx[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const int i2 = u + 8 * p;
        nx[p] = (i1y < N1 && i2 < N2) ? __ldcg(Wp + i1y * N2 + i2) : make_double2(0.0, 0.0);
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
                    nx[p] = (i1y < N1 && i2 < N2) ? __ldcg(Wp + cstride + i1y * N2 + i2) : make_double2(0.0, 0.0);
                }
            }
            fwd64_group(a, tw, sc, u);
            const int col = (i1y + u) & 31;
#pragma unroll
            for (int q = 0; q < 8; ++q) A[(8 * u + q) * 32 + col] = a[q];
        }
        __syncthreads();
#pragma unroll 1
        for (int round = 0; round < 2; ++round) {   // ---- x: forward, multiply by the coefficient spectrum, inverse
            const int r = (round * 8 + L.warp) * 4 + L.ln;
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

// ---- Z3: inverse z-FFT of 32 lines x 3 components + Green dyadic ------------------------------------------------------
// The [pos3][32 lines] tiles of W arrive by cp.async (L2 -> shared memory, no L1), double-buffered over the components;
// each group inverse-transforms its line, keeps the <= 4 x 3 kept outputs in registers and applies Eq. 4's dyadic
//   y_c = x_c - (k_b^2 F_c - k_c (k.F)) / (k.k - k_b^2),  k = k_inc + m o K  (unconjugated k.k)
// or Eq. 5's second cross product  y = x + (k x F) / (k.k - k_b^2).
template <bool HFORM>
static __device__ __forceinline__ void z3_item(const ApplyGeom& g, const cplx* Ws, const cplx* __restrict__ xb,
                                               cplx* __restrict__ yb, const double* __restrict__ kv, double k0, int tile,
                                               cplx* T0, cplx* T1, cplx* sc, const cplx* tw, const Lane64& L) {
    const int N3 = g.N3, NL = g.NL, u = L.u;
    const int l0 = tile * 32, line = L.warp * 4 + L.ln, l = l0 + line;
    auto load_tile = [&](cplx* T, int c) {
        const cplx* Wc = Ws + (long)c * 64 * NL + l0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int r = k * 8 + L.warp;
            const int ll = (L.lane - (r >> 3)) & 31;
            if (l0 + ll < NL) cp_async16_cg(&T[r * 32 + L.lane], Wc + (long)r * NL + ll);
        }
        cp_async_commit_();
    };
    load_tile(T0, 0);
    load_tile(T1, 1);
    const int col = (line + u) & 31;
    cplx F[3][4];
    cplx a[8];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (c < 2) cp_async_wait_<1>(); else cp_async_wait_<0>();
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
    if (l < NL) {
        const double kb2r = k0 * k0 * g.epsb_re, kb2i = k0 * k0 * g.epsb_im;
        const int i1 = l / g.N2, i2 = l - i1 * g.N2;
        const double k1 = kv[0] + (i1 + g.mmin[0]) * g.K[0];
        const double k2 = kv[1] + (i2 + g.mmin[1]) * g.K[1];
        const double k12 = k1 * k1 + k2 * k2;
        const long base = (long)l * N3;
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const int i3 = u + 8 * p;
            if (i3 >= N3) continue;
            const double k3 = kv[2] + (i3 + g.mmin[2]) * g.K[2];
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
                if (HFORM) {
                    const int c1 = c == 2 ? 0 : c + 1, c2 = c1 == 2 ? 0 : c1 + 1;
                    num = make_double2(-(kk[c1] * Fc[c2].x - kk[c2] * Fc[c1].x), -(kk[c1] * Fc[c2].y - kk[c2] * Fc[c1].y));
                } else {
                    num = cmul(kb2, Fc[c]);
                    num.x -= kk[c] * s.x;
                    num.y -= kk[c] * s.y;
                }
                const cplx q = cmul(num, rden);
                const cplx xv = xb[base + c * g.n + i3];
                yb[base + c * g.n + i3] = make_double2(xv.x - q.x, xv.y - q.y);
            }
        }
    }
}

// ---- the persistent kernel ------------------------------------------------------------------------------------------
struct Fused64Ctl {
    int* head;          // [1]    ticket counter               } zeroed by compact_active_kernel before every launch
    int* cnt;           // [3][maxB] items finished per solve  }
    int* nact;          // [1]    solves in the list
    int* list;          // [maxB] batch indices of the active solves, increasing
    const int* items;   // [ips]  slot pattern: (kind << 16) | index
    int ips, nlt, maxB;
};

template <bool HFORM>
__global__ void __launch_bounds__(F64_T, 2) apply_fused64_kernel(ApplyGeom g, const cplx* __restrict__ x,
                                                                 cplx* __restrict__ y, cplx* Wring,
                                                                 const double* __restrict__ kvec,
                                                                 const double* __restrict__ k0s, Fused64Ctl ctl) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* T0 = reinterpret_cast<cplx*>(smem_raw);   // [64][32]: XY plane / Z1 tile / Z3 tile 0
    cplx* T1 = T0 + 64 * 32;                        // Z3 tile 1
    cplx* scratch = T1 + 64 * 32;                   // [32 lines][SC_LINE]
    __shared__ int s_ticket;
    Lane64 L;
    L.lane = threadIdx.x & 31; L.warp = threadIdx.x >> 5; L.u = L.lane & 7; L.ln = L.lane >> 3;
    cplx tw[7];
    load_group_twiddles(tw, g.tw[0], L.u);          // all three axes are 64-point: one twiddle set
    cplx* sc = scratch + (L.warp * 4 + L.ln) * SC_LINE;
    const int nact = *ctl.nact;
    const int total = (nact + F64_LAG3) * ctl.ips;
    const long wslot = 3L * 64 * g.NL;
    int* cnt1 = ctl.cnt; int* cnt2 = ctl.cnt + ctl.maxB; int* cnt3 = ctl.cnt + 2 * ctl.maxB;
    if (threadIdx.x == 0) s_ticket = atomicAdd(ctl.head, 1);
    __syncthreads();
    int cur = s_ticket;
    while (cur < total) {
        int nxt = 0;
        if (threadIdx.x == 0) nxt = atomicAdd(ctl.head, 1);   // consumed after the item: the round trip is hidden
        const int slot = cur / ctl.ips;
        const int it = __ldg(ctl.items + (cur - slot * ctl.ips));
        const int kind = it >> 16, idx = it & 0xffff;
        const int p = slot - (kind == 0 ? 0 : kind == 1 ? F64_LAG2 : F64_LAG3);
        if (p >= 0 && p < nact) {
            const int b = ctl.list[p];
            cplx* Ws = Wring + (long)(p % F64_RING) * wslot;
            const cplx* xb = x + (long)b * 3 * g.n;
            if (kind == 0) {
                if (p >= F64_RING) wait_count(cnt3 + p - F64_RING, ctl.nlt);   // the ring slot's previous user is done
                z1_item<HFORM>(g, xb, Ws, kvec + 3 * b, idx, T0, sc, tw, L);
                signal_count(cnt1 + p);
            } else if (kind == 1) {
                wait_count(cnt1 + p, ctl.nlt);
                xy_item(g, Ws, idx, g.chat64, T0, sc, tw, L);
                signal_count(cnt2 + p);
            } else {
                wait_count(cnt2 + p, 64);
                z3_item<HFORM>(g, Ws, xb, y + (long)b * 3 * g.n, kvec + 3 * b, k0s[b], idx, T0, T1, sc, tw, L);
                signal_count(cnt3 + p);
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) s_ticket = nxt;
        __syncthreads();
        cur = s_ticket;
    }
}

// list of the solves still iterating (all of them when active == null), zeroed ticket counter and completion counters
__global__ void __launch_bounds__(1024) compact_active_kernel(const int* __restrict__ active, int batch, Fused64Ctl ctl) {
    __shared__ int wsum[32];
    __shared__ int base;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    if (t == 0) { base = 0; *ctl.head = 0; }
    for (int i = t; i < 3 * ctl.maxB; i += blockDim.x) ctl.cnt[i] = 0;
    __syncthreads();
    for (int b0 = 0; b0 < batch; b0 += blockDim.x) {
        const int b = b0 + t;
        const int f = b < batch && (!active || active[b]) ? 1 : 0;
        const unsigned m = __ballot_sync(0xffffffffu, f);
        if (lane == 0) wsum[warp] = __popc(m);
        __syncthreads();
        int off = base;
        for (int w = 0; w < warp; ++w) off += wsum[w];
        if (f) ctl.list[off + __popc(m & ((1u << lane) - 1))] = b;
        __syncthreads();
        if (t == 0) {
            int s = 0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += wsum[w];
            base += s;
        }
        __syncthreads();
    }
    if (t == 0) *ctl.nact = base;
}

static const size_t F64_SMEM = sizeof(cplx) * (2 * 64 * 32 + 32 * SC_LINE);

// host side -------------------------------------------------------------------------------------------------------------
size_t fused64_ring_elems(const ApplyGeom& g) { return (size_t)F64_RING * 3 * 64 * g.NL; }
int fused64_items_per_slot(const ApplyGeom& g) { return 2 * ((g.NL + 31) / 32) + 64; }

// slot pattern: the XY items and the two kinds of Z items spread evenly over the slot
void fused64_slot_pattern(const ApplyGeom& g, int* items) {
    const int nlt = (g.NL + 31) / 32, ips = 2 * nlt + 64;
    const int cnt[3] = {nlt, 64, nlt};
    int done[3] = {0, 0, 0};
    for (int k = 0; k < ips; ++k) {
        int best = -1;
        double bestpos = 2.0;
        for (int kind = 0; kind < 3; ++kind) {
            if (done[kind] >= cnt[kind]) continue;
            const double pos = (done[kind] + 0.5) / cnt[kind] + 1e-9 * kind;
            if (pos < bestpos) { bestpos = pos; best = kind; }
        }
        items[k] = (best << 16) | done[best];
        ++done[best];
    }
}

cudaError_t apply_fused64_init_attributes(int* grid_out) {
    cudaError_t e = cudaFuncSetAttribute(apply_fused64_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F64_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(apply_fused64_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F64_SMEM);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, per = 0;
    e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, apply_fused64_kernel<false>, F64_T, F64_SMEM);
    if (e == cudaSuccess) *grid_out = sms * (per > 0 ? per : 1);
    return e;
}

cudaError_t launch_apply_fused64(const ApplyGeom& g, int batch, const double* d_kvec, const double* d_k0, const cplx* d_x,
                                 cplx* d_y, const int* d_active, const Fused64Dev& f, cudaStream_t st) {
    Fused64Ctl ctl;
    ctl.head = f.head; ctl.cnt = f.cnt; ctl.nact = f.nact; ctl.list = f.list; ctl.items = f.items;
    ctl.nlt = (g.NL + 31) / 32; ctl.ips = 2 * ctl.nlt + 64; ctl.maxB = f.maxB;
    compact_active_kernel<<<1, 1024, 0, st>>>(d_active, batch, ctl);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    // enough CTAs for the items that can be in flight, never more than the persistent grid
    const long want = (long)(batch + F64_LAG3) * ctl.ips;
    const int grid = (int)(want < f.grid ? want : f.grid);
    if (g.hform) apply_fused64_kernel<true><<<grid, F64_T, F64_SMEM, st>>>(g, d_x, d_y, f.ring, d_kvec, d_k0, ctl);
    else apply_fused64_kernel<false><<<grid, F64_T, F64_SMEM, st>>>(g, d_x, d_y, f.ring, d_kvec, d_k0, ctl);
    return cudaGetLastError();
}

}  // namespace gsm
