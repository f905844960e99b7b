// arnoldi_cluster.cu - one Arnoldi step of GMRES with literal modified Gram-Schmidt ("GMRes ...
// according to Saad with the modified Gram-Schmidt orthogonalization"), each basis vector read from HBM ONCE.
//
//   for i = 0..j:  h_i = <v_i, w>;  w <- w - h_i v_i          (Saad Alg. 6.9, lines 4-7)
//   h_{j+1,j} = ||w||;  v_{j+1} = w / h_{j+1,j}               (lines 8-9), then the Givens update of the least squares
//
// One solve = one thread-block cluster.  The cluster keeps w on chip (registers, vlen / (CS * 256) complex numbers
// per thread) for the whole step.  Each v_i is streamed through shared memory exactly once: a 1-D bulk TMA copy
// (cp.async.bulk + mbarrier) brings CTA r's contiguous slice of v_i into one of two buffers while the previous
// slice is being used, the slice is dotted with w, the partial sums are exchanged through distributed shared memory
// (st.async + mbarrier, no cluster-wide barrier), and the same slice - read from shared memory once and held in
// registers across the exchange, so its buffer is refilled while the sums travel - updates w.  HBM traffic per step is
// (j + 3) V: read w, read v_0..v_j, write v_{j+1}; the paper's one-CUBLAS-call-per-dot/axpy schedule (made for a
// GTX Titan) moves 5 V per basis vector, the two-sweep fallback in krylov.cu 2 V.
//
// Reductions are deterministic: fixed-shape warp trees, then fixed-order sums over warps and over cluster ranks.
#include <cooperative_groups.h>
#include <cstdint>

#include "gsm_internal.cuh"
#include "krylov_device.cuh"

namespace cg = cooperative_groups;

namespace gsm {

#define MGS_T 256        // threads per CTA
#define MGS_E_LO 22      // complex elements of w per thread (registers): the kernel is instantiated for 22 (31^3: 5586 per
#define MGS_E_HI 24      // CTA) and 24 (32^3: 6144 per CTA, the most two slice buffers of a CTA leave room for)
#define MGS_MAXCS 16     // largest cluster (non-portable size, opt-in)
#define MGS_NW (MGS_T / 32)

static __device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
static __device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
static __device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
static __device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
// 1-D bulk copy global -> this CTA's shared memory, completion signalled on the mbarrier (bytes % 16 == 0)
static __device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

static __device__ __forceinline__ double warp_sum_x(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// address of the same shared-memory variable in CTA `rank` of the cluster (shared::cluster window)
static __device__ __forceinline__ uint32_t map_rank(uint32_t cta_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(cta_addr), "r"(rank));
    return r;
}
// 16-byte asynchronous store into a peer CTA's shared memory that also completes 16 bytes on the peer's mbarrier:
// the data is visible to whoever observes the mbarrier phase flip, with no cluster-wide barrier or fence.
static __device__ __forceinline__ void st_async_cplx(uint32_t remote_addr, cplx v, uint32_t remote_bar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 ::"r"(remote_addr), "d"(v.x), "d"(v.y), "r"(remote_bar) : "memory");
}

struct MgsSmem {
    uint64_t mbar[2];         // TMA completion of the two basis-slice buffers
    uint64_t rbar[2];         // arrival of the CS partial sums of an exchange (even / odd exchange number)
    cplx red[2][MGS_MAXCS];   // red[parity][rank]: per-CTA partial sums, written by every rank through DSMEM
    cplx wpart[MGS_NW];       // per-warp partial sums of this CTA
};

// Sum over the cluster of one complex number per thread; exchange number `step` (0, 1, 2, ... in program order).
// Every rank sends its CTA-level partial to all ranks with st.async, which completes bytes on the receiver's
// mbarrier; the receiver waits for CS * 16 bytes.  Exchanges alternate between two (mbarrier, buffer) pairs: rank X
// can only send exchange s+2 after it has received every rank's exchange s+1, which rank Y sends after all of its
// threads have consumed exchange s - so two pairs never collide.  All ranks sum the same values in the same fixed
// tree order: identical bits everywhere, deterministic.
static __device__ __forceinline__ void cluster_sum_send(MgsSmem* sm, cplx v, int step, unsigned cs, unsigned rank) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, par = step & 1;
    v.x = warp_sum_x(v.x);
    v.y = warp_sum_x(v.y);
    if (lane == 0) sm->wpart[warp] = v;
    __syncthreads();
    if (warp == 0) {
        if (lane == 0) mbar_expect_tx(&sm->rbar[par], cs * (uint32_t)sizeof(cplx));
        cplx t = make_double2(0.0, 0.0);
        if (lane < MGS_NW) t = sm->wpart[lane];
        t.x = warp_sum_x(t.x);
        t.y = warp_sum_x(t.y);
        if (lane < (int)cs)
            st_async_cplx(map_rank(smem_u32(&sm->red[par][rank]), lane), t, map_rank(smem_u32(&sm->rbar[par]), lane));
    }
}
static __device__ __forceinline__ cplx cluster_sum_recv(MgsSmem* sm, int step, unsigned cs) {
    const int par = step & 1;
    mbar_wait(&sm->rbar[par], (step >> 1) & 1);
    cplx q[MGS_MAXCS];
#pragma unroll
    for (int c = 0; c < MGS_MAXCS; ++c) q[c] = (c < (int)cs) ? sm->red[par][c] : make_double2(0.0, 0.0);
#pragma unroll
    for (int w = 1; w < MGS_MAXCS; w *= 2)
#pragma unroll
        for (int c = 0; c + w < MGS_MAXCS; c += 2 * w) { q[c].x += q[c + w].x; q[c].y += q[c + w].y; }
    return q[0];
}

// Persistent: grid = nclusters * CS CTAs (cluster = CS CTAs along x); cluster k runs solves k, k + nclusters, ...
// chunk = elements per CTA (<= MGS_T * MGS_E).  The first two basis slices of the NEXT solve are requested as soon as
// the last slice of the current one has been used, so the norm exchange, the write of v_{j+1}, the Givens update and
// the load of the next w all run under that transfer.
template <int MGS_E>
__global__ void __launch_bounds__(MGS_T, 1) arnoldi_mgs_kernel(KrylovDims d, KrylovState s, int batch, int j, int chunk) {
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned cs = cluster.num_blocks(), rank = cluster.block_rank();
    const int nclusters = gridDim.x / cs;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    cplx* vbuf0 = reinterpret_cast<cplx*>(smem_raw);
    cplx* vbuf1 = vbuf0 + chunk;
    cplx* hsm = vbuf1 + chunk;                                   // [ld]   h_0..h_j of this step
    cplx* snsm = hsm + d.ld;                                     // [mmax] previous rotations (rank 0 only)
    double* cssm = reinterpret_cast<double*>(snsm + d.mmax);     // [mmax]
    MgsSmem* sm = reinterpret_cast<MgsSmem*>(cssm + d.mmax + (d.mmax & 1));

    const int t = threadIdx.x;
    const long lo = (long)rank * chunk;
    const int len = (int)max(0L, min((long)chunk, d.vlen - lo));
    const uint32_t bytes = (uint32_t)len * (uint32_t)sizeof(cplx);
    const long vs = d.vstride ? d.vstride : (long)batch * d.vlen;

    if (t == 0) {
        mbar_init(&sm->mbar[0], 1);
        mbar_init(&sm->mbar[1], 1);
        mbar_init(&sm->rbar[0], 1);
        mbar_init(&sm->rbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // solves of this cluster that are still iterating (only this cluster ever changes their flags)
    auto next_active = [&](int from) {
        while (from < batch && !s.active[from]) from += nclusters;
        return from;
    };
    // j < 0: slot-refill scan, every solve is at its own Arnoldi index s.iters[b] (only this cluster changes it)
    auto index_of = [&](int bb) { return j >= 0 ? j : s.iters[bb]; };
    auto prefetch_first_two = [&](int bb) {   // thread 0 only
        const cplx* vb = s.basis + (long)bb * d.vlen + lo;
        mbar_expect_tx(&sm->mbar[0], bytes);
        bulk_g2s(vbuf0, vb, bytes, &sm->mbar[0]);
        if (index_of(bb) >= 1) {
            mbar_expect_tx(&sm->mbar[1], bytes);
            bulk_g2s(vbuf1, vb + vs, bytes, &sm->mbar[1]);
        }
    };
    int b = next_active((int)(blockIdx.x / cs));
    if (t == 0 && len > 0 && b < batch) prefetch_first_two(b);
    // every CTA of the cluster must have started (mbarriers initialised) before any remote write reaches it
    cluster.sync();

    uint32_t phase0 = 0, phase1 = 0;
    int xstep = 0;   // running exchange number of cluster_sum
    while (b < batch) {
        const int j = index_of(b);                                   // this solve's Arnoldi index
        const cplx* vb = s.basis + (long)b * d.vlen + lo;            // slice of v_0; v_i at + i * vs
        cplx* wg = s.basis + (long)b * d.vlen + (long)(j + 1) * vs + lo;
        if (rank == 0)
            for (int i = t; i < j; i += MGS_T) {
                cssm[i] = s.cs[(long)b * d.mmax + i];
                snsm[i] = s.sn[(long)b * d.mmax + i];
            }
        cplx w[MGS_E];
#pragma unroll
        for (int k = 0; k < MGS_E; ++k) {
            const int e = k * MGS_T + t;
            w[k] = (e < len) ? wg[e] : make_double2(0.0, 0.0);
        }
        const int bnext = next_active(b + nclusters);
        for (int i = 0; i <= j; ++i) {
            cplx* vbuf = (i & 1) ? vbuf1 : vbuf0;
            if (len > 0) {
                if (i & 1) { mbar_wait(&sm->mbar[1], phase1); phase1 ^= 1; }
                else       { mbar_wait(&sm->mbar[0], phase0); phase0 ^= 1; }
            }
            cplx acc = make_double2(0.0, 0.0);
            cplx v[MGS_E];   // the slice is read from shared memory once and kept for the update
#pragma unroll
            for (int k = 0; k < MGS_E; ++k) {   // conj(v) * w
                const int e = k * MGS_T + t;
                v[k] = (e < len) ? vbuf[e] : make_double2(0.0, 0.0);
                acc.x = fma(v[k].x, w[k].x, fma(v[k].y, w[k].y, acc.x));
                acc.y = fma(v[k].x, w[k].y, fma(-v[k].y, w[k].x, acc.y));
            }
            cluster_sum_send(sm, acc, xstep, cs, rank);   // contains a block barrier: every thread has read vbuf
            if (t == 32 && len > 0) {                     // so the buffer can be refilled while the sums travel
                if (i + 2 <= j) {
                    uint64_t* bar = &sm->mbar[i & 1];
                    mbar_expect_tx(bar, bytes);
                    bulk_g2s(vbuf, vb + (long)(i + 2) * vs, bytes, bar);
                } else if (i == j && bnext < batch) {
                    prefetch_first_two(bnext);   // both buffers are idle now
                }
            }
            const cplx h = cluster_sum_recv(sm, xstep++, cs);
#pragma unroll
            for (int k = 0; k < MGS_E; ++k) {   // w -= h v
                w[k].x = fma(-h.x, v[k].x, fma(h.y, v[k].y, w[k].x));
                w[k].y = fma(-h.x, v[k].y, fma(-h.y, v[k].x, w[k].y));
            }
            if (t == 0) hsm[i] = h;
        }
        cplx nn = make_double2(0.0, 0.0);
#pragma unroll
        for (int k = 0; k < MGS_E; ++k) nn.x = fma(w[k].x, w[k].x, fma(w[k].y, w[k].y, nn.x));
        cluster_sum_send(sm, nn, xstep, cs, rank);
        nn = cluster_sum_recv(sm, xstep++, cs);
        const double hn = sqrt(nn.x);
        const double sc = hn > 0.0 ? 1.0 / hn : 0.0;
#pragma unroll
        for (int k = 0; k < MGS_E; ++k) {
            const int e = k * MGS_T + t;
            if (e < len) wg[e] = make_double2(w[k].x * sc, w[k].y * sc);
        }
        if (rank == 0 && t == 0) givens_step(d, s, b, j, hsm, hn, cssm, snsm);
        __syncthreads();   // hsm / cssm / snsm are reused by the next solve
        b = bnext;
    }
    cluster.sync();   // no CTA leaves while a peer's asynchronous store to it could still be in flight
}

// the instantiation whose per-thread registers hold a CTA's slice of w
static const void* mgs_kernel_for(int chunk) {
    return chunk <= MGS_T * MGS_E_LO ? (const void*)arnoldi_mgs_kernel<MGS_E_LO> : (const void*)arnoldi_mgs_kernel<MGS_E_HI>;
}

size_t arnoldi_cluster_smem(const KrylovDims& d, int chunk) {
    return sizeof(cplx) * (2 * (size_t)chunk + d.ld + d.mmax) + sizeof(double) * (d.mmax + (d.mmax & 1)) +
           sizeof(MgsSmem) + 128;
}

// Smallest power-of-two cluster whose CTAs can each keep their slice of w in registers; 0 if the vector is too long
// or the device cannot co-schedule such a cluster (then krylov.cu's two-sweep path is used).
cudaError_t arnoldi_cluster_plan(const KrylovDims& d, int* cs_out, int* chunk_out, int* nclusters_out) {
    *nclusters_out = 0;
    *cs_out = 0;
    *chunk_out = 0;
    const long cap = (long)MGS_T * MGS_E_HI;
    int cs = 1;
    while (cs <= MGS_MAXCS && (d.vlen + cs - 1) / cs > cap) cs *= 2;
    if (cs > MGS_MAXCS) return cudaSuccess;
    const int chunk = (int)((d.vlen + cs - 1) / cs);
    const size_t smem = arnoldi_cluster_smem(d, chunk);
    if (smem > 227 * 1024) return cudaSuccess;
    // the attribute is per function, not per plan: always ask for the device maximum so that plans of different
    // sizes can coexist
    const void* kern = mgs_kernel_for(chunk);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    if (cs > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) { cudaGetLastError(); return cudaSuccess; }
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cs);
    cfg.blockDim = dim3(MGS_T);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int nclusters = 0;
    e = cudaOccupancyMaxActiveClusters(&nclusters, kern, &cfg);
    if (e != cudaSuccess || nclusters < 1) { cudaGetLastError(); return cudaSuccess; }
    *cs_out = cs;
    *chunk_out = chunk;
    *nclusters_out = nclusters;
    return cudaSuccess;
}

cudaError_t launch_arnoldi_cluster(const KrylovDims& d, const KrylovState& s, int batch, int j, int cs, int chunk,
                                   int nclusters, cudaStream_t st, Profiler* prof) {
    ProfScope ps_(prof, KC_ARNOLDI_MGS, st);   // (j + 3) V per solve still iterating, billed by run_batch afterwards
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(batch < nclusters ? batch : nclusters) * cs);
    cfg.blockDim = dim3(MGS_T);
    cfg.dynamicSmemBytes = arnoldi_cluster_smem(d, chunk);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cs;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    void* args[] = {(void*)&d, (void*)&s, (void*)&batch, (void*)&j, (void*)&chunk};
    return cudaLaunchKernelExC(&cfg, mgs_kernel_for(chunk), args);
}

}  // namespace gsm
