// nl_cluster.cuh -- the fused per-plane kernel SPREAD OVER A THREAD-BLOCK CLUSTER, for planes whose half-transformed
// form Z (Nx x 2 nky0 complex: 768 KiB at configs[2]) exceeds one SM's shared memory.
//
// Same steps as nl_fused2.cuh.  The batched kernels of nl_kernels.cuh send Z, P
// and the chi rows through HBM/L2 scratch (about 4x the algorithmic bytes; PAPER.md:84 is the 2013 version of that
// cost: transpose 17.9 % + extend 11.7 % of the GPU time spent moving data).  Here a cluster of C CTAs owns one plane
// at a time and the two x<->y hand-overs -- the "transpositions" of PAPER.md:61 -- are DISTRIBUTED SHARED MEMORY
// stores (st.shared::cluster) straight from the registers of the producing butterfly into the shared memory of the CTA
// that consumes the value; nothing but g, rhs and the real-space chi rows crosses L2/HBM.
//
// Decomposition (Nx = AX * BX, C = BX / 2 CTAs, so that a CTA owns AX row pairs and nky0 / C stored columns):
//   X1  CTA c runs the x-synthesis of ITS columns ky in [c CK, (c+1) CK), both stages, through a local exchange tile E
//       (the +ky and -ky transforms one after the other, so that E fits).  A stage-2 thread (column, k1) holds the
//       rows m = k1 + AX k2, k2 < BX, of its column: row pair q = k1 + AX (k2 mod C) belongs to CTA (k2 mod C), pair
//       storage k1 there -- it stores each value into that CTA's Zl (DSMEM), 128 B runs along cc.
//       The g columns of a CTA are ONE contiguous block of the plane: it is brought in by a 1-D bulk copy (TMA,
//       cp.async.bulk + mbarrier) issued a plane ahead by one thread.
//   --- barrier.cluster ---
//   Y   CTA c owns row pairs (m, m + Nx/2), m in [c AX, (c+1) AX); a WARP takes NPW of them and runs, with __syncwarp
//       only: pruned radix-AY + radix-8 to real space for the rows m, the same for the rows m + Nx/2 (one exchange
//       tile per pair, in place behind the pair storage), bracket with the chi rows, radix-8 + pruned-output
//       radix-AY back.  The spectral row P[pair][cc] goes from the registers of the last butterfly to the CTA that
//       owns column cc (DSMEM), 128 B runs.
//   --- barrier.cluster ---
//   X2  CTA c runs the x-analysis of its columns in place over the received P, deletes the padded modes, applies the
//       prefactor and adds to rhs.
// Measured on B200 (DESIGN.md sect. 6e): remote stores run at ~18 B/clk/SM whatever the form (st.shared::cluster,
// st.async, cp.async.bulk); a plane moves (C-1)/C x 1.5 Z through them.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "nl_fused2.cuh"

namespace gnl {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of `addr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, cplx v)
{
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1,%2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
// asynchronous 16-byte store into a peer's shared memory; completes `bytes` on the peer's mbarrier `bar` (both shared::cluster)
__device__ __forceinline__ void st_async(uint32_t addr, cplx v, uint32_t bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1,%2}, [%3];" ::"r"(addr),
                 "l"(__double_as_longlong(v.x)), "l"(__double_as_longlong(v.y)), "r"(bar) : "memory");
}
// Arrive on a peer's mbarrier WITHOUT a release fence: used where the arrive only tells the peer that this CTA's
// loads from a buffer have completed (their values are in registers), so there is nothing to publish.
__device__ __forceinline__ void mbar_arrive_remote_relaxed(uint32_t bar_cluster_addr)
{
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster_addr) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// ---- 1-D bulk copy global -> shared with mbarrier completion (TMA; SASS UBLKCP) ----
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "GNL_MBAR_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra GNL_MBAR_DONE_%=;\n\t"
        "bra GNL_MBAR_WAIT_%=;\n\t"
        "GNL_MBAR_DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
// wait without an acquire fence (no L1 invalidation): the waiter reads nothing that the arrivals published
__device__ __forceinline__ void mbar_wait_relaxed(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "GNL_MBARC_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.relaxed.cluster.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra GNL_MBARC_DONE_%=;\n\t"
        "bra GNL_MBARC_WAIT_%=;\n\t"
        "GNL_MBARC_DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar) : "memory");
}

template <int AX_, int BX_, int AY_, int NW_>
struct Clustered {
    static constexpr int AX = AX_, BX = BX_, AY = AY_, NW = NW_;
    static constexpr int NX = AX * BX, NY = 8 * AY, C = BX / 2;
    static constexpr int NKY0 = NY / 3, W2 = 2 * NKY0, NPAIR = NX / 2;
    static constexpr int M = NX / 3, NX0 = 2 * M;
    static constexpr int CK = NKY0 / C;        // stored columns per CTA
    static constexpr int PPC = NPAIR / C;      // row pairs per CTA (= AX)
    static constexpr int NPW = PPC / NW;       // row pairs per warp
    static constexpr int NT = 32 * NW;
    static constexpr int FY = AY * 9;          // y exchange tile of one row: [k1][9]
    // pair storage: row m + NX/2 at [0, W2), row m at [W2, 2 W2); the exchange tile starts at W2 (over row m, whose
    // values are in registers by then) and runs FY slots, past the end of the two rows
    static constexpr int PS = (W2 + FY) | 1;
    static constexpr int ZL = PPC * PS;
    // x exchange tile: both signs of the CK columns, HALF of the k1 range at a time (the stage-1 threads keep the other
    // half in registers), so that every thread has a stage-1 item and E still fits beside Zl
    static constexpr int BPX = Tile<AX, BX>::BP, AXH = AX / 2, CS = ((AXH * BPX) | 1) + ((((AXH * BPX) | 1) % 8 == 1) ? 4 : 0);
    static constexpr int E_CPLX = 2 * CK * CS;
    static constexpr int PLS = 2 * CK;         // P_local[pair][slot]: slot = column (+ky), CK + column (-ky)
    static constexpr int PL_CPLX = NPAIR * PLS;
    static constexpr int U_CPLX = E_CPLX > PL_CPLX ? E_CPLX : PL_CPLX;   // E and P_local share one region
    static constexpr int G_CPLX = CK * NX0;    // this CTA's columns of a g plane (one contiguous block)
    static constexpr int TWX = AX * BPX, TWY = AY * 9;
    static constexpr int NBAR = 3 + NW;        // mbarriers: g block, P_local full, U free, Zl rows of each warp full
    static constexpr int SMEM_CPLX = ZL + U_CPLX + G_CPLX + TWX + TWY + (NBAR + 2) / 2;   // + the edone counter
    static constexpr unsigned ZBYTES = NPW * 2 * W2 * 16;   // bytes a warp's pair storages receive per plane
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)SMEM_CPLX;
    static_assert(AX % 3 == 0 && AY % 3 == 0, "3/2 rule");
    static_assert(BX % 2 == 0 && NKY0 % C == 0 && PPC == AX, "C = BX/2 CTAs: a CTA owns AX row pairs and nky0/C columns");
    static_assert(PPC % NW == 0 && NPW * 8 <= 32 && AY <= 32, "a warp takes NPW pairs: NPW*8 lanes in Y1/Y3, AY lanes in Y2");
    static_assert(CK == 8, "P slots are swizzled over 8-slot halves; 128 B runs in both hand-overs");
    static_assert(2 * CK * BX == NT && 2 * CK * AXH <= NT && (2 * CK * AXH) % 32 == 0 && CK * AX <= NT && AX % 2 == 0,
                  "one item per thread in every x stage; whole warps in stage 2");
    static_assert((G_CPLX * 16) % 16 == 0, "bulk copy size");
};

template <int AX, int BX, int AY, int NW>
__global__ void __launch_bounds__(32 * NW, 1)
k_plane_cluster(const cplx* __restrict__ g, cplx* __restrict__ rhs, const cplx* __restrict__ R,
                const cplx* __restrict__ twx_g, const cplx* __restrict__ twy_g, int nz, int nv, int nslab,
                double kxmin, double kymin, double coef)
{
    using K = Clustered<AX, BX, AY, NW>;
    constexpr int NX = K::NX, NY = K::NY, C = K::C, NKY0 = K::NKY0, W2 = K::W2, NPAIR = K::NPAIR;
    constexpr int M = K::M, NX0 = K::NX0, CK = K::CK, PPC = K::PPC, NPW = K::NPW, NT = K::NT;
    constexpr int PS = K::PS, BPX = K::BPX, CS = K::CS, PLS = K::PLS;
    constexpr int AX1 = AX / 3, AY1 = AY / 3;
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(NKY0 == 8 * AY1, "the pruned radix-AY stage reads lo/hi thirds of nky0 = 8 AY/3 values");

    extern __shared__ cplx smem[];
    cplx* Zl = smem;                       // [PPC][PS]: the rows of this CTA's pairs (written by every CTA of the cluster)
    cplx* U = Zl + K::ZL;                  // E (x exchange tile) during X1 / P_local (written by every CTA) during Y, X2
    cplx* Gs = U + K::U_CPLX;              // this CTA's CK columns of the current g plane (bulk copy)
    cplx* twx = Gs + K::G_CPLX;            // W_NX^{n2 k1}, [k1][BPX]
    cplx* twy = twx + K::TWX;              // W_NY^{k1 k2}, [k1][9]
    const uint32_t bars = smem_u32(twy + K::TWY);
    const uint32_t gbar = bars, pfull = bars + 8, ufree = bars + 16, zfull0 = bars + 24;   // zfull of warp w: zfull0 + 8 w
    unsigned* edone = (unsigned*)(twy + K::TWY) + 2 * K::NBAR;   // stage-2 warps that have finished with E (this plane)

    const int tid = threadIdx.x;
    const int lane0 = tid & 31;
    const int warp = __shfl_sync(FULL, tid >> 5, 0);
    const uint32_t rank = cluster_ctarank();
    const int ncluster = gridDim.x / C, cl = blockIdx.x / C;
    const uint32_t zl_base = smem_u32(Zl), pl_base = smem_u32(U);
    const uint32_t pbytes = (uint32_t)(NPAIR * (2 * CK - (rank == 0 ? 1 : 0)) * sizeof(cplx));   // no -ky value for ky = 0

    load_twiddles_ab<AX, BX>(twx, twx_g);
    load_twiddles_ab<AY, 8>(twy, twy_g);
    if (tid == 0) {
        mbar_init(gbar, 1);
        mbar_init(pfull, 1);
        mbar_init(ufree, C);
        for (int w = 0; w < NW; ++w) mbar_init(zfull0 + 8 * w, 1);
        *edone = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const unsigned T = (unsigned)nslab * (unsigned)nz * (unsigned)nv;   // planes of this launch (< 2^31: checked by the host)
    const size_t plane_elems = (size_t)NX0 * NKY0;
    // planes are walked v-fastest so that neighbouring clusters share a chi plane in L2
    auto plane_of = [&](unsigned tt) {
        const unsigned v = tt % (unsigned)nv, zs = tt / (unsigned)nv;
        const unsigned z = zs % (unsigned)nz, sl = zs / (unsigned)nz;
        return (size_t)z + (size_t)nz * ((size_t)v + (size_t)nv * sl);
    };
    auto request_g = [&](unsigned tt) {   // one thread: this CTA's columns of plane tt -> Gs
        mbar_arrive_expect_tx(gbar, (uint32_t)(K::G_CPLX * sizeof(cplx)));
        bulk_g2s(smem_u32(Gs), g + plane_of(tt) * plane_elems + (size_t)rank * CK * NX0,
                 (uint32_t)(K::G_CPLX * sizeof(cplx)), gbar);
    };
    if (tid == 0 && (unsigned)cl < T) request_g((unsigned)cl);
    // every CTA of the cluster is resident and its mbarriers are initialised before anyone stores into it
    cluster_arrive();
    cluster_wait();

    // shared::cluster address of a peer's copy of a shared::cta address: that address plus a per-peer constant
    uint32_t peer[C];
#pragma unroll
    for (int r = 0; r < C; ++r) peer[r] = mapa_u32(zl_base, (uint32_t)r) - zl_base;

    // Synchronisation inside the plane loop is by mbarriers only (no cluster-wide barrier, so warps whose rows are
    // complete start while the stores of the others are still in flight):
    //   zfull[w]  (tx) the 2 W2 NPW values of warp w's pair storages have arrived            -> warp w starts Y
    //   ufree     (C arrivals) every CTA of the cluster has finished with its exchange tile E -> P may be pushed into U
    //   pfull     (tx) every P value of this CTA's columns has arrived                        -> X2
    // A sender is never more than one phase ahead of a receiver: plane p+1's rows are sent after the sender's pfull(p),
    // which every warp of every CTA completes only after its Y(p); plane p+1's P after zfull(p+1), which needs every
    // CTA's X1(p+1), which follows its X2(p).  (An mbarrier armed late tolerates one phase of early bytes, not two.)
    uint32_t ph = 0;
    for (unsigned t = (unsigned)cl; t < T; t += (unsigned)ncluster, ph ^= 1) {
        const size_t p = plane_of(t);
        const size_t q = (size_t)((t / (unsigned)nv) % (unsigned)nz) + (size_t)nz * (size_t)(t / ((unsigned)nv * (unsigned)nz));
        cplx* Rb = rhs + p * plane_elems + (size_t)rank * CK * NX0;
        const cplx* Rc = R + q * ((size_t)NX * NY);
        if (tid == 0) mbar_arrive_expect_tx(pfull, pbytes);
        if (lane0 == 0) mbar_arrive_expect_tx(zfull0 + 8 * warp, K::ZBYTES);
        {  // pull the next plane's rhs columns of this CTA towards L2 while this one is being worked on
            const unsigned tn = t + (unsigned)ncluster;
            if (tn < T) {
                const char* b = (const char*)(rhs + plane_of(tn) * plane_elems + (size_t)rank * CK * NX0);
                for (size_t off = (size_t)tid * 128; off < (size_t)CK * NX0 * sizeof(cplx); off += (size_t)NT * 128)
                    prefetch_l2(b + off);
            }
        }

        // =============== X1: derivative, pad, x-synthesis of this CTA's columns; rows go to their owners ===============
        mbar_wait(gbar, ph);
        if (rank == 0) {   // Hermitian part of the ky = 0 column (reading R7), in place in the staged block
            if (tid > 0 && tid < NX0 / 2) {
                const cplx a = Gs[tid], b = Gs[NX0 - tid];
                Gs[tid] = cmake(0.5 * (a.x + b.x), 0.5 * (a.y - b.y));
                Gs[NX0 - tid] = cmake(0.5 * (a.x + b.x), 0.5 * (b.y - a.y));
            } else if (tid == 0) {
                Gs[0].y = 0.0;
            }
            __syncthreads();
        }
        {
            // stage 1, every thread: column-sign c2 = (sign, column), position n2: pruned radix-AX over n1 (i = n2 + BX n1),
            // twiddle W_NX^{n2 k1}.  The k1 < AX/2 half goes to E now, the other half after the first stage-2 pass.
            const int n2 = opaque(tid % BX), c2 = opaque(tid / BX);
            cplx out[AX];
            {
                const int col1 = c2 % CK;
                const cplx* Fc = Gs + col1 * NX0 + n2;
                const double ky = kymin * (double)((int)rank * CK + col1), dn2 = (double)n2;
                const double kys = (c2 / CK) ? ky : -ky;  // (i kx - ky) F for +ky, (i kx + ky) F for -ky
                cplx lo[AX1], hi[AX1];
#pragma unroll
                for (int a = 0; a < AX1; ++a) {
                    lo[a] = deriv_mul(Fc[BX * a], kxmin * (dn2 + (double)(BX * a)), kys);                // i = n2 + BX a      (kx >= 0)
                    hi[a] = deriv_mul(Fc[BX * a + M], kxmin * (dn2 + (double)(BX * a + M - NX0)), kys);  // i = n2 + BX a + M  (kx < 0)
                }
                if (n2 == 0) hi[0] = cmake(0.0, 0.0);  // i = M: the Nyquist row is ignored (R6)
                dft_pruned_in<AX, +1>(lo, hi, out);
#pragma unroll
                for (int k1 = 1; k1 < AX; ++k1) {
                    const cplx w = twx[k1 * BPX + n2];
                    out[k1] = cmul(out[k1], w.x, w.y);
                }
            }
            __syncthreads();   // every thread has read its g values
            if (tid == 0 && t + (unsigned)ncluster < T) request_g(t + (unsigned)ncluster);   // the next plane's block, a plane ahead
#pragma unroll
            for (int hk = 0; hk < 2; ++hk) {
                {
                    cplx* Ec = U + c2 * CS + n2;
#pragma unroll
                    for (int k1 = 0; k1 < K::AXH; ++k1) Ec[k1 * BPX] = out[hk * K::AXH + k1];
                }
                __syncthreads();
                if (tid < 2 * CK * K::AXH) {
                    // stage 2: radix-BX over n2 for fixed k1; row m = k1 + AX k2 -> CTA k2 mod C, pair storage k1.
                    // Lanes run over the 2 CK column-signs: two 128 B runs per store instruction and k1 value.
                    const int c2s = tid % (2 * CK), k1 = hk * K::AXH + tid / (2 * CK);
                    const int sg = c2s / CK, kyi = (int)rank * CK + c2s % CK;
                    const bool zero = (sg == 1 && kyi == 0);  // there is no -0 column: slot cc = nky0 holds zeros
                    cplx v[BX];
                    const cplx* Ec = U + c2s * CS + (k1 - hk * K::AXH) * BPX;
#pragma unroll
                    for (int i = 0; i < BX; ++i) v[i] = zero ? cmake(0.0, 0.0) : Ec[i];
                    Dft<BX, +1>::run(v);
                    const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
                    const uint32_t a0 = zl_base + (uint32_t)((k1 * PS + cc) * sizeof(cplx));
                    const uint32_t zb = zfull0 + 8 * (uint32_t)(k1 / NPW);   // the warp that owns pair k1 at the receiver
                    const double sgn = sg ? -1.0 : 1.0;                      // -ky columns hold the conjugate
#pragma unroll
                    for (int k2 = 0; k2 < BX; ++k2) {
                        // half 0 (row m < NX/2) sits at [W2, 2 W2), half 1 at [0, W2)
                        st_async(a0 + (uint32_t)((k2 < C ? W2 : 0) * sizeof(cplx)) + peer[k2 % C],
                                 cmake(v[k2].x, sgn * v[k2].y), zb + peer[k2 % C]);
                    }
                    if (hk == 1) {
                        // The last stage-2 warp to get here tells every CTA of the cluster that this CTA's U may
                        // receive P from now on (all loads from E have completed: their values went into the stores).
                        // No CTA barrier: the warps without a stage-2 item are already waiting for their rows.
                        __syncwarp(FULL);
                        if (lane0 == 0 && atomicAdd(edone, 1u) == (unsigned)(2 * CK * K::AXH / 32 - 1)) {
                            *edone = 0;
#pragma unroll
                            for (int r = 0; r < C; ++r) mbar_arrive_remote_relaxed(ufree + peer[r]);
                        }
                    }
                }
                if (hk == 0) __syncthreads();  // E is free for the second half
            }
        }
        // chi rows of this warp's first pair, requested while the rows arrive
        const int lane = opaque(lane0);
        const int k1y = lane < AY ? lane : lane - AY;   // lanes >= AY shadow an item (same addresses) and skip the stores
        const bool act2 = lane < AY;
        cplx chv[8];
        {
            const int m = (int)rank * PPC + warp * NPW;
            const cplx* Rr = Rc + (size_t)m * NY + k1y;
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) chv[k2] = ldg_nc_early(Rr + AY * k2);
        }
        mbar_wait(zfull0 + 8 * warp, ph);

        // =============== Y: this warp's NPW row pairs, __syncwarp only ===============
        {
            const int j1 = (lane >> 3) < NPW ? (lane >> 3) : 0;   // Y1 / Y3 item: pair j1 of the warp, position lane & 7
            const bool act1 = (lane >> 3) < NPW;
            const int n2 = lane & 7;
            cplx* Zw = Zl + (warp * NPW) * PS;                    // this warp's pair storages
            cplx tq[8];
#pragma unroll
            for (int k2 = 1; k2 < 8; ++k2) tq[k2] = twy[k1y * 9 + k2];
            double nlx[NPW][8];                                   // bracket of the rows m (first halves), kept in registers
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                {  // Y1: pruned radix-AY of rows m (h = 0: second half of the storage) / m + NX/2 (h = 1: first half)
                    const cplx* Zr = Zw + j1 * PS + (h ? 0 : W2) + n2;
                    cplx lo[AY1], hi[AY1];
#pragma unroll
                    for (int a = 0; a < AY1; ++a) {
                        lo[a] = Zr[8 * a];
                        hi[a] = Zr[8 * a + NKY0];
                    }
                    cplx out[AY];
                    dft_pruned_in<AY, +1>(lo, hi, out);
                    __syncwarp(FULL);  // h = 0: rows m are in registers before the tiles overwrite them; h = 1: Y2 done
                    if (act1) {
                        cplx* tile = Zw + j1 * PS + W2 + n2;
#pragma unroll
                        for (int k1 = 0; k1 < AY; ++k1) tile[k1 * 9] = out[k1];
                    }
                }
                __syncwarp(FULL);
#pragma unroll
                for (int j = 0; j < NPW; ++j) {  // Y2: twiddle + radix-8 to real space, bracket; pair j, k1 = lane
                    // chi rows of the NEXT item (pair j+1 of this half, or pair 0 of the second half), requested before
                    // this item's butterflies so that their latency hides behind them
                    cplx chn[8];
                    const int jn = (j + 1 < NPW) ? j + 1 : 0, hn = (j + 1 < NPW) ? h : 1;
                    if (!(h == 1 && j + 1 == NPW)) {
                        const int m = (int)rank * PPC + warp * NPW + jn + hn * NPAIR;
                        const cplx* Rr = Rc + (size_t)m * NY + k1y;
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2) chn[k2] = ldg_nc_early(Rr + AY * k2);
                    }
                    cplx* tile = Zw + j * PS + W2 + k1y * 9;
                    cplx v[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) v[i] = tile[i];
                    dft8_twiddled<+1>(v, tq);   // (dx g + i dy g)(row, y = k1 + AY k2)
                    if (h == 0) {
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2) nlx[j][k2] = fma(chv[k2].x, v[k2].y, -chv[k2].y * v[k2].x);
                    } else {
                        cplx w[8];
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2)
                            w[k2] = cmake(nlx[j][k2], fma(chv[k2].x, v[k2].y, -chv[k2].y * v[k2].x));
                        Dft<8, -1>::run(w);
#pragma unroll
                        for (int k2 = 1; k2 < 8; ++k2) w[k2] = cmul(w[k2], tq[k2].x, -tq[k2].y);
                        if (act2) {  // own slots of the tile: no other lane reads or writes them in this phase
#pragma unroll
                            for (int k2 = 0; k2 < 8; ++k2) tile[k2] = w[k2];
                        }
                    }
                    if (!(h == 1 && j + 1 == NPW)) {
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2) chv[k2] = chn[k2];
                    }
                }
                __syncwarp(FULL);
            }
            {  // Y3: pruned-output radix-AY; P[pair][cc] goes to the CTA that owns column cc
                const cplx* tile = Zw + j1 * PS + W2 + n2;
                cplx in[AY];
#pragma unroll
                for (int n1 = 0; n1 < AY; ++n1) in[n1] = tile[n1 * 9];
                cplx lo[AY1], hi[AY1];
                dft_pruned_out<AY, -1>(in, lo, hi);
                mbar_wait_relaxed(ufree, ph);   // every CTA of the cluster is done with its exchange tile
                if (act1) {
                    const int qg = (int)rank * PPC + warp * NPW + j1;   // global pair index = row of P_local
                    const uint32_t row = pl_base + (uint32_t)(qg * PLS * sizeof(cplx));
                    const int sw = (int)rank & 7;                        // slot swizzle of this sender's rows (qg / AX)
#pragma unroll
                    for (int c = 0; c < AY1; ++c) {
                        {  // +ky half: ky = n2 + 8 c
                            const int ky = n2 + 8 * c;
                            st_async(row + (uint32_t)(((ky % CK) ^ sw) * sizeof(cplx)) + peer[c], lo[c], pfull + peer[c]);
                        }
                        {  // -ky half: cc = nky0 + n2 + 8 c  <->  ky = nky0 - n2 - 8 c (ky = nky0 is a deleted mode)
                            const int ky = NKY0 - n2 - 8 * c;
                            const uint32_t dl = n2 ? peer[C - 1 - c] : peer[(C - c) % C];   // owner ky / CK
                            if (ky < NKY0)
                                st_async(row + (uint32_t)((CK + ((ky % CK) ^ sw)) * sizeof(cplx)) + dl, hi[c], pfull + dl);
                        }
                    }
                }
            }
        }
        // rhs values of this thread's share of X2 stage 2, requested while the P rows arrive
        cplx r0[AX1], r1[AX1];
        const int k2s = tid % BX, cols = (tid / BX) % CK;
        if (tid < CK * BX) {
            const cplx* Rcol = Rb + (size_t)cols * NX0 + k2s;
#pragma unroll
            for (int c = 0; c < AX1; ++c) {
                r0[c] = ldg_early(Rcol + BX * c);
                r1[c] = ldg_early(Rcol + BX * c + M);
            }
        }
        mbar_wait(pfull, ph);

        // =============== X2: x-analysis of this CTA's columns in place over P_local; delete modes, prefactor, add ===============
        cplx* Pl = U;
        if (tid < CK * AX) {  // stage 1: unpack the row pair, radix-BX over n2 for fixed n1 (m = n1 + AX n2), twiddle
            const int col = tid % CK, n1 = tid / CK;
            const int kyi = (int)rank * CK + col;
            cplx x[BX];
#pragma unroll
            for (int n2 = 0; n2 < C; ++n2) {
                const cplx* Pr = Pl + (n1 + AX * n2) * PLS;
                const cplx pp = Pr[col ^ n2];
                const cplx pm = kyi ? Pr[CK + (col ^ n2)] : pp;
                x[n2] = cmake(pp.x + pm.x, pp.y - pm.y);          // 2 N^_m  = P+ + conj P-
                x[n2 + C] = cmake(pp.y + pm.y, pm.x - pp.x);      // 2 N^_m' = -i (P+ - conj P-)
            }
            Dft<BX, -1>::run(x);
#pragma unroll
            for (int k2 = 0; k2 < BX; ++k2) {  // tile slot (col, n1, k2) replaces P[n1 + AX (k2 mod C)][half k2 / C]
                const cplx w = twx[n1 * BPX + k2];
                Pl[(n1 + AX * (k2 % C)) * PLS + CK * (k2 / C) + (col ^ (k2 % C))] = (k2 == 0) ? x[0] : cmul(x[k2], w.x, -w.y);
            }
        }
        __syncthreads();
        if (tid < CK * BX) {  // stage 2: pruned-output radix-AX over n1 for fixed k2; i = k2 + BX c
            const int k2 = k2s, col = cols;
            cplx in[AX];
            const cplx* Pc = Pl + (AX * (k2 % C)) * PLS + CK * (k2 / C) + (col ^ (k2 % C));
#pragma unroll
            for (int n1 = 0; n1 < AX; ++n1) in[n1] = Pc[n1 * PLS];
            cplx lo[AX1], hi[AX1];
            dft_pruned_out<AX, -1>(in, lo, hi);
            cplx* Rcol = Rb + (size_t)col * NX0 + k2;
#pragma unroll
            for (int c = 0; c < AX1; ++c) {
                Rcol[BX * c] = cmake(fma(coef, lo[c].x, r0[c].x), fma(coef, lo[c].y, r0[c].y));
                if (c != 0 || k2 != 0)  // i = M is the Nyquist row: untouched (R6)
                    Rcol[BX * c + M] = cmake(fma(coef, hi[c].x, r1[c].x), fma(coef, hi[c].y, r1[c].y));
            }
        }
        __syncthreads();  // P_local is consumed before the next plane's E overwrites it
    }
    // no CTA leaves while a peer may still store into it
    cluster_arrive();
    cluster_wait();
}

}  // namespace gnl
