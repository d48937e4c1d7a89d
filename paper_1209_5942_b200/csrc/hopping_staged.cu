// hopping_staged.cu -- staged variants of the hopping kernel (rows a1-a7 of SURVEY.md section 8(a),
// eq. 6), selected by lqcd_set_hop_variant; the default stays the plain kernel of
// hopping.cu.  BASELINE.json's north_star asks for "neighbour spinors staged through shared memory
// or TMA" with every choice evidenced by counters: these are the variants those counters were taken
// on (profiles/r02_hopping_staged.md).  Same arithmetic, same order of operations per site as the
// plain kernel, so the parity tests run unchanged on every variant.
//
// Variant 1..3, "link ring" (depth D = variant): the links of a site are read exactly once by exactly
// one thread, so nothing is gained by a cache -- but in the plain kernel the 9 x 16 bytes of a link
// occupy 18 registers from the moment the load is issued, and 168 registers hold about one hop of
// loads in flight.  Here every thread owns D slots of 144 bytes in shared memory and fetches the link
// of hop h + D with cp.async (LDGSTS: global -> shared, no register) while it works on hop h, whose
// link it reads back with LDS.128.  In flight per thread: D links in shared memory plus whatever
// spinor loads ptxas schedules ahead in the registers the links no longer need.
//
// Variant 4, 5, "bulk": in the grouped layout the forward link U_mu(x) of a warp's 32 sites is ONE contiguous block
// (4608 bytes in double/18), so lane 0 of every warp fetches it with a single bulk-asynchronous copy (cp.async.bulk,
// global -> shared, completion counted on the warp's own mbarrier) at the start of the kernel; the hop waits on the
// barrier and reads its link with LDS.128.  Variant 4 stages the z and t links, variant 5 all four directions.
// Backward links and all spinors take the plain path.
#include "site_ops.cuh"

namespace lqcd {
namespace {

template <typename T, int RECON> struct LinkBytes {
    static constexpr int n16 = (RECON * (int)sizeof(T)) / 16;            // whole 16-byte elements per link
    static constexpr int tail8 = ((RECON * (int)sizeof(T)) % 16) / 8;    // float/18: one trailing float2
    static constexpr int slot = (n16 + tail8) * 16;                      // bytes per thread and slot
    static constexpr int group = RECON * (int)sizeof(T) * 32;            // bytes per group of 32 links
};

// No "memory" clobbers: the ring is only ever touched through these volatile asm statements, which keep their order
// among themselves, and the kernel reads no global memory it writes.  A clobber would pin every LDG of a hop behind
// that hop's wait_group, i.e. forbid ptxas the software pipelining of the spinor loads the plain kernel lives on.
__device__ __forceinline__ void cp_async16(unsigned dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async8(unsigned dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(dst), "l"(src));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ double2 lds128d(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ float4 lds128f(unsigned addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];\n" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float2 lds64f(unsigned addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

// issue the copy of link (par, mu, idx) into the thread's slot at shared address `dst` ([element][thread])
template <typename T, int RECON>
__device__ __forceinline__ void link_fetch(unsigned dst, const void* gauge, int G, int par, int mu, int idx) {
    typedef LinkBytes<T, RECON> LB;
    const char* p = reinterpret_cast<const char*>(gauge) + gauge_block(par, mu, G, idx >> 5) * LB::group;
#pragma unroll
    for (int j = 0; j < LB::n16; ++j) cp_async16(dst + j * (LQCD_HOP_MAX_THREADS * 16), p + j * 512 + (idx & 31) * 16);
    if (LB::tail8) cp_async8(dst + LB::n16 * (LQCD_HOP_MAX_THREADS * 16), p + LB::n16 * 512 + (idx & 31) * 8);
}

// read the link back from the slot
template <int RECON>
__device__ __forceinline__ void link_read(unsigned slot, double (&u)[18]) {
#pragma unroll
    for (int j = 0; j < RECON / 2; ++j) {
        const double2 v = lds128d(slot + j * (LQCD_HOP_MAX_THREADS * 16));
        u[2 * j] = v.x;
        u[2 * j + 1] = v.y;
    }
    if (RECON == 12) reconstruct_row2(u);
}
template <int RECON>
__device__ __forceinline__ void link_read(unsigned slot, float (&u)[18]) {
    constexpr int n16 = RECON / 4;
#pragma unroll
    for (int j = 0; j < n16; ++j) {
        const float4 v = lds128f(slot + j * (LQCD_HOP_MAX_THREADS * 16));
        u[4 * j] = v.x; u[4 * j + 1] = v.y; u[4 * j + 2] = v.z; u[4 * j + 3] = v.w;
    }
    if (RECON == 18) {
        const float2 w = lds64f(slot + n16 * (LQCD_HOP_MAX_THREADS * 16));
        u[16] = w.x;
        u[17] = w.y;
    } else {
        reconstruct_row2(u);
    }
}

template <typename T, int RECON, int MU, int FWD, int DAG>
__device__ __forceinline__ void hop_from_slot(T (&acc)[24], const HopArgs& a, const T (&u)[18], int e_nb, bool wrap) {
    constexpr int S = (FWD ? -1 : +1) * (DAG ? -1 : +1);
    T psi[24], h[12], chi[12];
    load_spinor(a.in, e_nb, psi);
    project<MU, S>(psi, h);
    if (FWD) su3_mul(u, h, chi);
    else     su3_dag_mul(u, h, chi);
    // the staged variants cover lattices with real boundary phases only (hopping_variant_covers): the phase is the sign
    // of the accumulation, as in the default kernel's REALPH build, and the thread has no branch
    accumulate_scaled<MU, S>(acc, chi, wrap ? (T)a.g.ph_re[MU] : (T)1);
}

template <typename T, int RECON, int DAG, int MODE, int D, int NB>
__global__ void __launch_bounds__(LQCD_HOP_MAX_THREADS, NB) hopping_ring_kernel(const HopArgs a) {
    typedef LinkBytes<T, RECON> LB;
    extern __shared__ __align__(16) unsigned char ring[];   // [D][element][thread]
    if (a.scal != nullptr && a.scal->done) return;
    const int Vh = a.g.Vh;
    const int blk = a.reverse ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
    const int e = blk * blockDim.x + threadIdx.x;
    if (e < Vh) {
        const int N0h = a.g.N0h, N1 = a.g.N1, N2 = a.g.N2, N3 = a.g.N3;
        int x0h, x1, x2, x3;
        site_coords(a.g, e, x0h, x1, x2, x3);
        const int r = (x1 + x2 + x3 + a.out_parity) & 1;
        const int s1 = N0h, s2 = N0h * N1, s3 = N0h * N1 * N2;
        // hop h = 2 mu + (backward): neighbour index and wrap flag
        int nb[8];
        bool wr[8];
        wr[0] = (r == 1) && (x0h == N0h - 1); nb[0] = wr[0] ? e - (N0h - 1) : e + r;
        wr[1] = (r == 0) && (x0h == 0);       nb[1] = wr[1] ? e + (N0h - 1) : e + r - 1;
        wr[2] = (x1 == N1 - 1); nb[2] = wr[2] ? e - (N1 - 1) * s1 : e + s1;
        wr[3] = (x1 == 0);      nb[3] = wr[3] ? e + (N1 - 1) * s1 : e - s1;
        wr[4] = (x2 == N2 - 1); nb[4] = wr[4] ? e - (N2 - 1) * s2 : e + s2;
        wr[5] = (x2 == 0);      nb[5] = wr[5] ? e + (N2 - 1) * s2 : e - s2;
        wr[6] = (x3 == N3 - 1); nb[6] = wr[6] ? e - (N3 - 1) * s3 : e + s3;
        wr[7] = (x3 == 0);      nb[7] = wr[7] ? e + (N3 - 1) * s3 : e - s3;

        const unsigned ring0 = (unsigned)__cvta_generic_to_shared(ring) + threadIdx.x * 16;
        constexpr int SLOT = LB::slot * LQCD_HOP_MAX_THREADS;   // bytes per slot of the whole CTA
        // forward link: (out_parity, mu, e); backward link: (other parity, mu, neighbour)
#define LQCD_FETCH(H)                                                                                          \
        link_fetch<T, RECON>(ring0 + ((H) % D) * SLOT, a.gauge, a.g.G, ((H) & 1) ? 1 - a.out_parity : a.out_parity, \
                             (H) >> 1, ((H) & 1) ? nb[H] : e)
#pragma unroll
        for (int h = 0; h < D; ++h) { LQCD_FETCH(h); cp_async_commit(); }

        T acc[24];
        if (MODE >= 1) {
            T x[24];
            load_spinor(a.aux, e, x);
            const T dur = (T)a.ep.du_re, dui = (T)a.ep.du_im, ddr = (T)a.ep.dd_re, ddi = (T)a.ep.dd_im;
#pragma unroll
            for (int c = 0; c < 12; ++c) {
                const T dr = (c < 6) ? dur : ddr, di = (c < 6) ? dui : ddi;
                acc[2 * c] = fma_(-di, x[2 * c + 1], dr * x[2 * c]);
                acc[2 * c + 1] = fma_(di, x[2 * c], dr * x[2 * c + 1]);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = 0;
        }

        // hop H: wait until its link has landed (at most D - 1 younger copies may still be in flight), read it,
        // hand the slot to hop H + D, then do the arithmetic
#define LQCD_HOP(H)                                                                           \
        {                                                                                     \
            cp_async_wait<D - 1>();                                                           \
            T u[18];                                                                          \
            link_read<RECON>(ring0 + ((H) % D) * SLOT, u);                                    \
            if ((H) + D < 8) { LQCD_FETCH(((H) + D) & 7); }                                   \
            cp_async_commit();                                                                \
            hop_from_slot<T, RECON, ((H) >> 1), (1 - ((H) & 1)), DAG>(acc, a, u, nb[H], wr[H]);   \
        }
        LQCD_HOP(0) LQCD_HOP(1) LQCD_HOP(2) LQCD_HOP(3) LQCD_HOP(4) LQCD_HOP(5) LQCD_HOP(6) LQCD_HOP(7)
#undef LQCD_HOP
#undef LQCD_FETCH

        T o[24];
        const T cur = (T)a.ep.cu_re, cui = (T)a.ep.cu_im, cdr = (T)a.ep.cd_re, cdi = (T)a.ep.cd_im;
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            const T cr = (c < 6) ? cur : cdr, ci = (c < 6) ? cui : cdi;
            o[2 * c] = fma_(-ci, acc[2 * c + 1], cr * acc[2 * c]);
            o[2 * c + 1] = fma_(ci, acc[2 * c], cr * acc[2 * c + 1]);
        }
        store_spinor(a.out, e, o);
    } else if (e < a.g.G * 32) {   // pad sites of the last group hold zeros
        T z[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) z[i] = 0;
        store_spinor(a.out, e, z);
    }
}

template <typename T, int RECON, int D, int NB>
cudaError_t launch_ring(int dagger, int mode, const HopArgs& a, int block, cudaStream_t st) {
    const int grid = (a.g.Vh + block - 1) / block;
    const size_t smem = (size_t)D * LinkBytes<T, RECON>::slot * LQCD_HOP_MAX_THREADS;
#define LQCD_RING_CASE(DG, M)                                                                             \
    if (dagger == DG && mode == M) {                                                                      \
        auto k = hopping_ring_kernel<T, RECON, DG, M, D, NB>;                                             \
        if (smem > 48 * 1024) {                                                                           \
            cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
            if (e != cudaSuccess) return e;                                                               \
        }                                                                                                 \
        k<<<grid, block, smem, st>>>(a);                                                                  \
        return cudaGetLastError();                                                                        \
    }
    LQCD_RING_CASE(0, 0) LQCD_RING_CASE(0, 1) LQCD_RING_CASE(1, 0) LQCD_RING_CASE(1, 1)
#undef LQCD_RING_CASE
    return cudaErrorInvalidValue;
}

template <int D>
cudaError_t launch_ring_fmt(int precision, int recon, int dagger, int mode, const HopArgs& a, int block, cudaStream_t st) {
    if (precision == 0) {
        return recon == 12 ? launch_ring<double, 12, D, 4>(dagger, mode, a, block, st)
                           : launch_ring<double, 18, D, 3>(dagger, mode, a, block, st);
    }
    return recon == 12 ? launch_ring<float, 12, D, 7>(dagger, mode, a, block, st)
                       : launch_ring<float, 18, D, 3>(dagger, mode, a, block, st);
}


// ------------------------------------------------------------------------------------------------ variants 4, 5: bulk
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::);
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes));
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar));
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity));
}

// the link of this lane out of a staged group block ([element][lane], the global layout of one group)
template <int RECON>
__device__ __forceinline__ void block_read(unsigned blk, double (&u)[18]) {
#pragma unroll
    for (int j = 0; j < RECON / 2; ++j) {
        const double2 v = lds128d(blk + j * 512);
        u[2 * j] = v.x;
        u[2 * j + 1] = v.y;
    }
    if (RECON == 12) reconstruct_row2(u);
}
template <int RECON>
__device__ __forceinline__ void block_read(unsigned blk, float (&u)[18]) {
    constexpr int n16 = RECON / 4;
#pragma unroll
    for (int j = 0; j < n16; ++j) {
        const float4 v = lds128f(blk + j * 512);
        u[4 * j] = v.x; u[4 * j + 1] = v.y; u[4 * j + 2] = v.z; u[4 * j + 3] = v.w;
    }
    if (RECON == 12) reconstruct_row2(u);   // 18: the trailing float2 plane (8 bytes per lane) is read by the caller
}

template <typename T, int RECON, int DAG, int MODE, int NMU, int NB>
__global__ void __launch_bounds__(LQCD_HOP_MAX_THREADS, NB) hopping_bulk_kernel(const HopArgs a) {
    typedef LinkBytes<T, RECON> LB;
    constexpr int MU0 = 4 - NMU;                       // staged directions MU0..3
    extern __shared__ __align__(128) unsigned char stage[];   // [warp][staged mu][group block], then one mbarrier per warp
    if (a.scal != nullptr && a.scal->done) return;
    const int Vh = a.g.Vh;
    const int blk = a.reverse ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
    const int e = blk * blockDim.x + threadIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nwarps = LQCD_HOP_MAX_THREADS / 32;
    const unsigned stage0 = (unsigned)__cvta_generic_to_shared(stage) + warp * (NMU * LB::group);
    const unsigned bar = (unsigned)__cvta_generic_to_shared(stage) + nwarps * (NMU * LB::group) + warp * 8;
    const bool warp_live = (e >> 5) < a.g.G;           // whole warp: same group
    if (lane == 0) {
        mbar_init(bar, 1);
        if (warp_live) {
            mbar_expect_tx(bar, NMU * LB::group);
#pragma unroll
            for (int m = 0; m < NMU; ++m) {
                const char* src = reinterpret_cast<const char*>(a.gauge) +
                                  gauge_block(a.out_parity, MU0 + m, a.g.G, e >> 5) * LB::group;
                bulk_g2s(stage0 + m * LB::group, src, LB::group, bar);
            }
        }
    }
    __syncwarp();
    if (e < Vh) {
        const int N0h = a.g.N0h, N1 = a.g.N1, N2 = a.g.N2, N3 = a.g.N3;
        int x0h, x1, x2, x3;
        site_coords(a.g, e, x0h, x1, x2, x3);
        const int r = (x1 + x2 + x3 + a.out_parity) & 1;
        const int s1 = N0h, s2 = N0h * N1, s3 = N0h * N1 * N2;
        int nb[8];
        bool wr[8];
        wr[0] = (r == 1) && (x0h == N0h - 1); nb[0] = wr[0] ? e - (N0h - 1) : e + r;
        wr[1] = (r == 0) && (x0h == 0);       nb[1] = wr[1] ? e + (N0h - 1) : e + r - 1;
        wr[2] = (x1 == N1 - 1); nb[2] = wr[2] ? e - (N1 - 1) * s1 : e + s1;
        wr[3] = (x1 == 0);      nb[3] = wr[3] ? e + (N1 - 1) * s1 : e - s1;
        wr[4] = (x2 == N2 - 1); nb[4] = wr[4] ? e - (N2 - 1) * s2 : e + s2;
        wr[5] = (x2 == 0);      nb[5] = wr[5] ? e + (N2 - 1) * s2 : e - s2;
        wr[6] = (x3 == N3 - 1); nb[6] = wr[6] ? e - (N3 - 1) * s3 : e + s3;
        wr[7] = (x3 == 0);      nb[7] = wr[7] ? e + (N3 - 1) * s3 : e - s3;

        T acc[24];
        if (MODE >= 1) {
            T x[24];
            load_spinor(a.aux, e, x);
            const T dur = (T)a.ep.du_re, dui = (T)a.ep.du_im, ddr = (T)a.ep.dd_re, ddi = (T)a.ep.dd_im;
#pragma unroll
            for (int c = 0; c < 12; ++c) {
                const T dr = (c < 6) ? dur : ddr, di = (c < 6) ? dui : ddi;
                acc[2 * c] = fma_(-di, x[2 * c + 1], dr * x[2 * c]);
                acc[2 * c + 1] = fma_(di, x[2 * c], dr * x[2 * c + 1]);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = 0;
        }
        bool waited = false;
#define LQCD_HOP(H)                                                                                              \
        {                                                                                                        \
            T u[18];                                                                                             \
            if (((H) & 1) == 0 && ((H) >> 1) >= MU0) {   /* staged forward link */                               \
                if (!waited) { mbar_wait(bar, 0); waited = true; }                                               \
                const unsigned b = stage0 + (((H) >> 1) - MU0) * LB::group;                                      \
                block_read<RECON>(b + lane * 16, u);                                                             \
                if (sizeof(T) == 4 && RECON == 18) {                                                             \
                    const float2 w = lds64f(b + 4 * 512 + lane * 8);                                             \
                    u[16] = (T)w.x; u[17] = (T)w.y;                                                              \
                }                                                                                                \
            } else {                                                                                             \
                load_link<RECON>(a.gauge, a.g.G, ((H) & 1) ? 1 - a.out_parity : a.out_parity, (H) >> 1,          \
                                 ((H) & 1) ? nb[H] : e, u);                                                      \
            }                                                                                                    \
            hop_from_slot<T, RECON, ((H) >> 1), (1 - ((H) & 1)), DAG>(acc, a, u, nb[H], wr[H]);                  \
        }
        LQCD_HOP(0) LQCD_HOP(1) LQCD_HOP(2) LQCD_HOP(3) LQCD_HOP(4) LQCD_HOP(5) LQCD_HOP(6) LQCD_HOP(7)
#undef LQCD_HOP

        T o[24];
        const T cur = (T)a.ep.cu_re, cui = (T)a.ep.cu_im, cdr = (T)a.ep.cd_re, cdi = (T)a.ep.cd_im;
#pragma unroll
        for (int c = 0; c < 12; ++c) {
            const T cr = (c < 6) ? cur : cdr, ci = (c < 6) ? cui : cdi;
            o[2 * c] = fma_(-ci, acc[2 * c + 1], cr * acc[2 * c]);
            o[2 * c + 1] = fma_(ci, acc[2 * c], cr * acc[2 * c + 1]);
        }
        store_spinor(a.out, e, o);
    } else {
        if (e < a.g.G * 32) {   // pad sites of the last group hold zeros
            T z[24];
#pragma unroll
            for (int i = 0; i < 24; ++i) z[i] = 0;
            store_spinor(a.out, e, z);
        }
        if (warp_live) mbar_wait(bar, 0);   // the copy targets this CTA's shared memory: it must land before the CTA ends
    }
}

template <typename T, int RECON, int NMU, int NB>
cudaError_t launch_bulk(int dagger, int mode, const HopArgs& a, cudaStream_t st) {
    const int block = LQCD_HOP_MAX_THREADS;   // the staging area is laid out for four warps
    const int grid = (a.g.Vh + block - 1) / block;
    const size_t smem = (size_t)(block / 32) * (NMU * LinkBytes<T, RECON>::group + 8);
#define LQCD_BULK_CASE(DG, M)                                                                             \
    if (dagger == DG && mode == M) {                                                                      \
        auto k = hopping_bulk_kernel<T, RECON, DG, M, NMU, NB>;                                           \
        if (smem > 48 * 1024) {                                                                           \
            cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
            if (e != cudaSuccess) return e;                                                               \
        }                                                                                                 \
        k<<<grid, block, smem, st>>>(a);                                                                  \
        return cudaGetLastError();                                                                        \
    }
    LQCD_BULK_CASE(0, 0) LQCD_BULK_CASE(0, 1) LQCD_BULK_CASE(1, 0) LQCD_BULK_CASE(1, 1)
#undef LQCD_BULK_CASE
    return cudaErrorInvalidValue;
}

template <int NMU>
cudaError_t launch_bulk_fmt(int precision, int recon, int dagger, int mode, const HopArgs& a, cudaStream_t st) {
    if (precision == 0) {
        return recon == 12 ? launch_bulk<double, 12, NMU, 4>(dagger, mode, a, st)
                           : launch_bulk<double, 18, NMU, 3>(dagger, mode, a, st);
    }
    return recon == 12 ? launch_bulk<float, 12, NMU, 7>(dagger, mode, a, st)
                       : launch_bulk<float, 18, NMU, 3>(dagger, mode, a, st);
}

}  // namespace

bool hopping_variant_covers(int variant, int mode, const Geometry& g, const SiteRange* range) {
    return variant >= 1 && variant <= 5 && mode <= 1 && !g.slab && range == nullptr && g.real_ph;
}

cudaError_t launch_hopping_variant(int variant, int precision, int recon, int dagger, int mode, const Geometry& g,
                                   const Epilogue& ep, const void* gauge, const void* in, void* out, const void* aux,
                                   int out_parity, int reverse, CgScalars* scal, int block, cudaStream_t st) {
    HopArgs a;
    a.rg.base = 0; a.rg.count = g.Vh; a.rg.n1 = g.Vh; a.rg.skip = 0;
    a.reverse = reverse;
    a.gauge = gauge; a.in = in; a.out = out; a.aux = aux; a.dotw = nullptr; a.dotw2 = nullptr;
    a.g = g; a.ep = ep; a.out_parity = out_parity; a.red.partials = nullptr; a.scal = scal;
    a.tile_gy = a.tile_n2h = 0;
    a.general_phases = 0;
    if (block <= 0 || block > LQCD_HOP_MAX_THREADS || (block % 32) != 0) block = LQCD_HOP_MAX_THREADS;
    count_launch();
    ProfScope prof(mode, st);
    switch (variant) {
        case 1: return launch_ring_fmt<1>(precision, recon, dagger, mode, a, block, st);
        case 2: return launch_ring_fmt<2>(precision, recon, dagger, mode, a, block, st);
        case 3: return launch_ring_fmt<3>(precision, recon, dagger, mode, a, block, st);
        case 4: return launch_bulk_fmt<2>(precision, recon, dagger, mode, a, st);
        case 5: return launch_bulk_fmt<4>(precision, recon, dagger, mode, a, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace lqcd
