// nl_group.cuh -- the fused per-plane kernel for planes beyond one SM, spread over a GROUP of G co-resident CTAs whose
// x<->y hand-overs go through a small per-group scratch that lives in the 126 MB L2.
//
// Same steps and the same phase structure as nl_cluster.cuh, changed where the
// measurements of that kernel pointed (DESIGN.md sect. 6e): distributed-shared-memory stores run at 18 B/clk/SM, in
// series with the butterflies, and only 15 clusters of 8 CTAs are co-resident on the 148 SMs.  Here
//   * a group is G consecutive CTAs of one cooperative launch (any G that divides the work; no placement constraint,
//     every SM is used), one plane per group at a time;
//   * the half-transformed arrays Z[pair][m+Nx/2 | m][cc] and P[pair][cc] of the group's CURRENT plane sit in global
//     memory, 1.1 MB per group at 384 x 192: written and read again within microseconds and overwritten by the next
//     plane, so the lines never leave L2 (HBM sees g, rhs and the chi rows only);
//   * rows come back for the y transforms as ONE 1-D bulk copy (TMA, cp.async.bulk + mbarrier) per row pair, straight
//     into the warp's pair storage; g column blocks come in the same way, a block ahead;
//   * the two hand-overs of a plane are ordered by two counters per group in global memory (release: bar.sync +
//     __threadfence + atomicAdd by one thread; acquire: one thread polls, bar.sync), monotonic over the launch.
// Phases per plane and CTA r of the group (Nx = AX * BX, Ny = 8 AY):
//   X1  column units u = r, r + G, ... (8 stored columns each): derivative, pad, pruned radix-AX, radix-BX, rows to Z
//   Y   row pairs [r PPG, (r+1) PPG): a warp takes NPW pairs at a time and runs, with __syncwarp only, pruned radix-AY +
//       radix-8 to real space (rows m, then rows m + Nx/2, one exchange tile per pair behind its rows), the bracket
//       with the chi rows, radix-8 + pruned-output radix-AY back; P rows go to global memory from registers
//   X2  column units again: unpack the row pair, radix-BX, pruned-output radix-AX, delete modes, prefactor, rhs +=
// Scratch reads bypass L1 (ld.global.cg / TMA): L1 is not coherent across SMs and the addresses repeat every plane.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "nl_cluster.cuh"

namespace gnl {

__device__ __forceinline__ cplx ldg_cg(const cplx* p)   // L2 only
{
    cplx v;
    asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// L2 eviction priorities: the per-group scratch is written and read again within microseconds, every plane (keep it:
// evict_last); g streams through once (evict_first), so that the scratch lines are not the ones that leave L2
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// Drop a 128-byte line from L2 without writing it back: the scratch rows a warp has just pulled into shared memory are
// dead (the next plane overwrites them in full), so their dirty lines need never reach HBM.
__device__ __forceinline__ void l2_discard_line(const void* p)
{
    asm volatile("discard.global.L2 [%0], 128;" ::"l"(p) : "memory");
}
__device__ __forceinline__ void stg_hint(cplx* p, cplx v, uint64_t pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ cplx ldg_cg_hint(const cplx* p, uint64_t pol)   // L2 only
{
    cplx v;
    asm volatile("ld.global.cg.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol) : "memory");
    return v;
}
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}

// NH: k1 passes of the X1 exchange tile (2: half of the k1 range at a time, for AX = 24; 1 for AX = 12).
// CHIV: chi per plane (chi_has_v = 1): chi goes through X1 like g and its rows are transformed next to those of g in Y
// (no real-space chi array R); else chi is shared over v and its real-space rows (dx chi, dy chi) come from R.
// BY: radix of the second y stage (Ny = AY * BY; 8, or 16 for Ny = 384); NPW: row pairs per warp item (NPW * BY <= 32).
// AX2 x BX2: the split of Nx used by the x-analysis (X2) when it differs from the synthesis' (768 = 48 x 16 on the way in,
// 24 x 32 on the way back: every thread has an item in the stage that carries the pruned radix).
// CK: stored columns per column unit (8: 128 B runs in both hand-overs; 4: 64 B runs, for CTAs of 4 warps, two per SM).
template <int AX_, int BX_, int AY_, int G_, int NW_, int NH_, bool CHIV_, int BY_ = 8, int NPW_ = 3, int AX2_ = 0, int BX2_ = 0,
          int CK_ = 8>
struct Grouped {
    static constexpr int AX2 = AX2_ ? AX2_ : AX_, BX2 = BX2_ ? BX2_ : BX_, C22 = BX2 / 2;
    static constexpr int BPX2 = Tile<AX2, BX2>::BP;
    static constexpr int AX = AX_, BX = BX_, AY = AY_, G = G_, NW = NW_, NH = NH_, BY = BY_, BYP = BY_ + 1;
    static constexpr bool CHIV = CHIV_;
    static constexpr int NF = CHIV ? 2 : 1;            // fields that go through X1 and the row hand-over
    static constexpr int NX = AX * BX, NY = BY * AY, C2 = BX / 2;
    static constexpr int NKY0 = NY / 3, W2 = 2 * NKY0, NPAIR = NX / 2;
    static constexpr int M = NX / 3, NX0 = 2 * M;
    static constexpr int CK = CK_;                     // stored columns per unit
    static constexpr int NUNIT = NKY0 / CK;            // column units per plane
    static constexpr int UPC = NUNIT / G_;             // column units per CTA
    static constexpr int PPG = NPAIR / G;              // row pairs per CTA
    static constexpr int NPW = NPW_;                   // row pairs per warp item
    static constexpr int NITEM = PPG / NPW;            // items per CTA
    static constexpr int NT = 32 * NW;
    static constexpr int FY = AY * BYP;                // y exchange tile of one row: [k1][BY + 1]
    static constexpr int PS = (W2 + FY) | 1;           // pair storage: rows m + NX/2 | m, the tile over row m and beyond
    static constexpr int YB_CPLX = NW * NF * NPW * PS;
    static constexpr int BPX = Tile<AX, BX>::BP, AXH = AX / NH;
    static constexpr int CSH = ((AXH * BPX) | 1) + ((((AXH * BPX) | 1) % 8 == 1) ? 4 : 0);   // tile of one column-sign, AXH values of k1
    static constexpr int E_CPLX = 2 * CK * CSH;        // X1: both signs of a unit's columns, AXH values of k1 at a time
    static constexpr int CSF = Tile<AX2, BX2>::STRIDE;
    static constexpr int XBIG = AX2 > BX2 ? AX2 : BX2;
    static constexpr int UPP0 = NT / (CK * XBIG);
    static constexpr int UPP = UPP0 < 1 ? 1 : (UPP0 < UPC ? UPP0 : UPC);   // X2: units per pass
    static constexpr int TX_CPLX = UPP * CK * CSF;     // X2: exchange tiles of the units of one pass
    static constexpr int XR_CPLX = E_CPLX > TX_CPLX ? E_CPLX : TX_CPLX;
    static constexpr int G_CPLX = CK * NX0;            // one unit's columns of a spectral plane (one contiguous block)
    static constexpr int TWX = AX * BPX, TWY = AY * BYP;
    static constexpr int TWX2 = (AX2 == AX && BX2 == BX) ? 0 : AX2 * BPX2;   // X2's own twiddle table when its split differs
    static constexpr int NBAR = 1 + NW;                // mbarriers: column block, rows of each warp
    // With several k1 passes (NH > 1) the odd passes of X1 use a SECOND exchange tile E1 behind the first, so that the
    // stores of pass hk + 1 need not wait for the stage-2 reads of pass hk: one CTA barrier per pass instead of two.  Its
    // column-sign stride is the smallest odd one that holds AXH rows (the last row needs BX slots, not BPX).  Taken when
    // the kernel still fits shared memory with the staged column block moved behind both tiles.
    static constexpr int CSH1 = ((AXH - 1) * BPX + BX) | 1;
    static constexpr int E1_OFF = E_CPLX;
    static constexpr int E2_CPLX = E_CPLX + 2 * CK * CSH1;
    static constexpr int GS_OFF_DB = XR_CPLX > E2_CPLX ? XR_CPLX : E2_CPLX;
    static constexpr int A_CPLX_DB = YB_CPLX > GS_OFF_DB + G_CPLX ? YB_CPLX : GS_OFF_DB + G_CPLX;
    static constexpr bool EDB = NH_ > 1 && sizeof(cplx) * (size_t)(A_CPLX_DB + TWX + TWX2 + TWY + (NBAR + 1) / 2) <= 227 * 1024;
    // One region A serves the phases in turn: X1 (E at 0, E1 behind it, the staged column block behind the x tiles), Y (the
    // warps' pair storages: no block is in flight then), X2 (Tx at 0, the next plane's first block behind it).
    static constexpr int GS_OFF = EDB ? GS_OFF_DB : XR_CPLX;
    static constexpr int A_CPLX = YB_CPLX > GS_OFF + G_CPLX ? YB_CPLX : GS_OFF + G_CPLX;
    static constexpr int SMEM_CPLX = A_CPLX + TWX + TWX2 + TWY + (NBAR + 1) / 2;
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)SMEM_CPLX;
    static constexpr int MINB = (NW <= 4 && SMEM_BYTES <= 113 * 1024) ? 2 : 1;   // CTAs per SM the kernel is built for
    static constexpr size_t ZS_CPLX = (size_t)NPAIR * 2 * W2, PS_CPLX = (size_t)NPAIR * W2;   // per-group scratch
    static constexpr size_t GROUP_SCRATCH_CPLX = NF * ZS_CPLX + PS_CPLX;
    // consumed scratch lines are dropped from L2 where the scratch of all groups (148 SMs) exceeds what L2 keeps; a
    // compile-time choice: at 384 x 192 the mere presence of the code costs 5 % (what ptxas hoists changes)
    static constexpr bool DISCARD = GROUP_SCRATCH_CPLX * sizeof(cplx) * (148 / G_) > ((size_t)64 << 20);
    static_assert(AX % 3 == 0 && AY % 3 == 0 && AX % NH == 0 && BX % 2 == 0, "3/2 rule; k1 passes; row pairs");
    static_assert(NKY0 % CK == 0 && NUNIT % G == 0 && NPAIR % G == 0 && PPG % NPW == 0, "the group divides the work");
    static_assert(NPW * BY <= 32 && AY <= 32 && NKY0 == BY * (AY / 3) && (BY == 8 || BY == 16), "lanes of the y stages");
    static_assert(2 * CK * BX <= NT && 2 * CK * AXH <= NT && UPP >= 1 && UPC % UPP == 0, "one item per thread in every x stage");
    static_assert(AX2 * BX2 == NX && AX2 % 3 == 0 && BX2 % 2 == 0 && UPP * CK * BX2 <= NT, "the x-analysis split");
};

// grid = groups * G CTAs (cooperative launch: every CTA is resident).  scratch: groups * GROUP_SCRATCH_CPLX values;
// cnt: 2 * groups counters, zeroed before the launch.  chi: the spectral chi planes when CHIV (laid out like g), else
// unused; R: the real-space chi rows when !CHIV, else unused.
// EM (!CHIV only): chi = phi_bar - v_par A_par_bar composed in real space, by linearity: R holds the
// real-space fields of phi_bar, R2 those of A_par_bar (one plane per (z, slab) each), vp[v + nv * species] the v_par
// coefficients; slab sl of the launch is global slab slab0 + sl = w + nw * species.
template <int AX, int BX, int AY, int G, int NW, int NH, bool CHIV, bool EM = false, int BY = 8, int NPW_ = 3, int AX2_ = 0, int BX2_ = 0,
          int CK_ = 8>
__global__ void __launch_bounds__(32 * NW, (Grouped<AX, BX, AY, G, NW, NH, CHIV, BY, NPW_, AX2_, BX2_, CK_>::MINB))
k_plane_group(const cplx* __restrict__ g, cplx* __restrict__ rhs, const cplx* __restrict__ R, const cplx* __restrict__ chi,
              const cplx* __restrict__ twx_g, const cplx* __restrict__ twy_g, cplx* __restrict__ scratch,
              unsigned* __restrict__ cnt, int nz, int nv, int nslab, double kxmin, double kymin, double coef,
              const cplx* __restrict__ R2 = nullptr, const double* __restrict__ vp = nullptr, int nw = 1, int slab0 = 0)
{
    static_assert(!(EM && CHIV), "the composition needs chi-like fields shared over v");
    using K = Grouped<AX, BX, AY, G, NW, NH, CHIV, BY, NPW_, AX2_, BX2_, CK_>;
    constexpr int BYP = K::BYP, AX2 = K::AX2, BX2 = K::BX2, C22 = K::C22, BPX2 = K::BPX2, AX21 = K::AX2 / 3;
    constexpr int NX = K::NX, NY = K::NY, C2 = K::C2, NKY0 = K::NKY0, W2 = K::W2, NPAIR = K::NPAIR, NF = K::NF;
    constexpr int M = K::M, NX0 = K::NX0, CK = K::CK, PPG = K::PPG, NPW = K::NPW, NT = K::NT, UPC = K::UPC, UPP = K::UPP;
    constexpr int PS = K::PS, BPX = K::BPX, CSH = K::CSH, CSF = K::CSF, AXH = K::AXH;
    constexpr int AX1 = AX / 3, AY1 = AY / 3;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr uint32_t GBYTES = (uint32_t)(K::G_CPLX * sizeof(cplx));

    extern __shared__ cplx smem[];
    cplx* A = smem;                        // X1: E / X2: Tx / Y: pair storages of the warps
    cplx* Gs = A + K::GS_OFF;              // a unit's columns of g or chi (bulk copy), behind the x tiles
    cplx* twx = A + K::A_CPLX;             // W_NX^{n2 k1}, [k1][BPX]
    cplx* twx2 = K::TWX2 ? twx + K::TWX : twx;   // W_NX^{n1 k2} of the x-analysis split, [n1][BPX2]
    cplx* twy = twx + K::TWX + K::TWX2;    // W_NY^{k1 k2}, [k1][BY + 1]
    const uint32_t bars = smem_u32(twy + K::TWY);
    const uint32_t gbar = bars;

    const int tid = threadIdx.x;
    const int lane0 = tid & 31;
    const int warp = __shfl_sync(FULL, tid >> 5, 0);
    const uint32_t ybar = bars + 8 + 8 * (uint32_t)warp;
    const int ngroup = gridDim.x / G, grp = blockIdx.x / G, rank = blockIdx.x % G;
    cplx* Zs = scratch + (size_t)grp * K::GROUP_SCRATCH_CPLX;   // [field][pair][row m + NX/2 | row m][cc]; field 0 = g
    cplx* Ps = Zs + NF * K::ZS_CPLX;                            // [pair][cc]
    unsigned* zcnt = cnt + 2 * grp;
    unsigned* pcnt = zcnt + 1;

    load_twiddles_ab<AX, BX>(twx, twx_g);
    if constexpr (K::TWX2 != 0) load_twiddles_ab<AX2, BX2>(twx2, twx_g);
    load_twiddles_ab<AY, BY>(twy, twy_g);
    if (tid == 0) {
        mbar_init(gbar, 1);
        for (int w = 0; w < NW; ++w) mbar_init(bars + 8 + 8 * w, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const unsigned T = (unsigned)nslab * (unsigned)nz * (unsigned)nv;   // planes of this launch (< 2^31: checked by the host)
    const size_t plane_elems = (size_t)NX0 * NKY0;
    // planes are walked v-fastest so that neighbouring groups share a chi plane in L2
    auto plane_of = [&](unsigned tt) {
        const unsigned v = tt % (unsigned)nv, zs = tt / (unsigned)nv;
        const unsigned z = zs % (unsigned)nz, sl = zs / (unsigned)nz;
        return (size_t)z + (size_t)nz * ((size_t)v + (size_t)nv * sl);
    };
    const uint64_t pol_keep = l2_policy_evict_last(), pol_stream = l2_policy_evict_first();
    // X1 step s of a plane: field s / UPC (with CHIV: chi first, then g), column unit rank + G (s mod UPC)
    auto request_block = [&](unsigned tt, int s) {   // one thread: the 8 columns of step s of plane tt -> Gs
        const cplx* src = (CHIV && s < UPC) ? chi : g;
        mbar_arrive_expect_tx(gbar, GBYTES);
        bulk_g2s_hint(smem_u32(Gs), src + plane_of(tt) * plane_elems + (size_t)(rank + G * (s % UPC)) * CK * NX0, GBYTES, gbar,
                      pol_stream);
    };
    if (tid == 0 && (unsigned)grp < T) request_block((unsigned)grp, 0);

    uint32_t gph = 0, yph = 0;
    unsigned it = 0;
    for (unsigned t = (unsigned)grp; t < T; t += (unsigned)ngroup, ++it) {
        const size_t p = plane_of(t);
        const size_t q = (size_t)((t / (unsigned)nv) % (unsigned)nz) + (size_t)nz * (size_t)(t / ((unsigned)nv * (unsigned)nz));
        cplx* Rb = rhs + p * plane_elems;
        [[maybe_unused]] const cplx* Rc = CHIV ? nullptr : R + q * ((size_t)NX * NY);
        [[maybe_unused]] const cplx* Rc2 = EM ? R2 + q * ((size_t)NX * NY) : nullptr;
        [[maybe_unused]] double vpar = 0.0;
        if constexpr (EM) vpar = __ldg(vp + (t % (unsigned)nv) + (unsigned)nv * (((unsigned)slab0 + t / ((unsigned)nv * (unsigned)nz)) / (unsigned)nw));

        // =============== X1: derivative, pad, x-synthesis of this CTA's column units; rows go to Z ===============
#pragma unroll 1
        for (int s = 0; s < NF * UPC; ++s) {
            const int unit = rank + G * (s % UPC);
            cplx* Zf = Zs + ((CHIV && s < UPC) ? K::ZS_CPLX : 0);   // field 0 = g, field 1 = chi
            mbar_wait(gbar, gph);
            gph ^= 1;
            if (unit == 0) {   // Hermitian part of the ky = 0 column (reading R7), in place in the staged block
                if (tid > 0 && tid < NX0 / 2) {
                    const cplx a = Gs[tid], b = Gs[NX0 - tid];
                    Gs[tid] = cmake(0.5 * (a.x + b.x), 0.5 * (a.y - b.y));
                    Gs[NX0 - tid] = cmake(0.5 * (a.x + b.x), 0.5 * (b.y - a.y));
                } else if (tid == 0) {
                    Gs[0].y = 0.0;
                }
                __syncthreads();
            }
            // stage 1: column-sign c2 = (sign, column), position n2: pruned radix-AX over n1 (i = n2 + BX n1), twiddle
            // W_NX^{n2 k1}.  AXH values of k1 go to E at a time, the rest waits in registers.
            const int n2 = opaque(tid % BX), c2 = opaque(tid / BX);
            const bool has1 = tid < 2 * CK * BX;
            cplx out[AX];
            if (has1) {
                const int col1 = c2 % CK;
                const cplx* Fc = Gs + col1 * NX0 + n2;
                const double ky = kymin * (double)(unit * CK + col1), dn2 = (double)n2;
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
            __syncthreads();   // every thread has read its values of the block
            // the next step's block (the first block of the next plane is requested when X2 starts: region A holds
            // the pair storages in between)
            if (tid == 0 && s + 1 < NF * UPC) request_block(t, s + 1);
#pragma unroll
            for (int hk = 0; hk < K::NH; ++hk) {
                // odd passes go through the second tile when there is one (K::EDB)
                const int eoff = (K::EDB && (hk & 1)) ? K::E1_OFF : 0, csh = (K::EDB && (hk & 1)) ? K::CSH1 : CSH;
                if (has1) {
                    cplx* Ec = A + eoff + c2 * csh + n2;
#pragma unroll
                    for (int k1 = 0; k1 < AXH; ++k1) Ec[k1 * BPX] = out[hk * AXH + k1];
                }
                __syncthreads();
                if (tid < 2 * CK * AXH) {
                    // stage 2: radix-BX over n2 for fixed k1; row m = k1 + AX k2 is half k2 / C2 of pair k1 + AX (k2 mod C2).
                    // Lanes run over the 2 CK column-signs: two 128 B runs per store instruction and k1 value.
                    const int c2s = tid % (2 * CK), k1 = hk * AXH + tid / (2 * CK);
                    const int sg = c2s / CK, kyi = unit * CK + c2s % CK;
                    const bool zero = (sg == 1 && kyi == 0);  // there is no -0 column: slot cc = nky0 holds zeros
                    cplx v[BX];
                    const cplx* Ec = A + eoff + c2s * csh + (k1 - hk * AXH) * BPX;
#pragma unroll
                    for (int i = 0; i < BX; ++i) v[i] = zero ? cmake(0.0, 0.0) : Ec[i];
                    Dft<BX, +1>::run(v);
                    const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
                    cplx* Zc = Zf + (size_t)k1 * (2 * W2) + cc;
                    const double sgn = sg ? -1.0 : 1.0;   // -ky columns hold the conjugate
#pragma unroll
                    for (int k2 = 0; k2 < BX; ++k2)      // pair storage: row m + NX/2 (k2 >= C2) first, then row m
                        stg_hint(Zc + (size_t)(AX * (k2 % C2)) * (2 * W2) + (k2 < C2 ? W2 : 0), cmake(v[k2].x, sgn * v[k2].y), pol_keep);
                }
                // E is free for the next step (and, with one tile, for the next k1 pass).  With two tiles the barrier of
                // pass hk + 1 already separates the stage-2 reads of pass hk from the stores of pass hk + 2 into the same tile.
                if (!K::EDB || hk == K::NH - 1) __syncthreads();
            }
        }
        // ---- hand-over 1: every CTA of the group has written its columns of Z (a group of one: the CTA barrier that
        // ended X1 has ordered the stores; no counter) ----
        if constexpr (G > 1) {
            if (tid == 0) {
                __threadfence();
                atomicAdd(zcnt, 1u);
                while (ld_acquire_gpu(zcnt) < (unsigned)G * (it + 1)) {}
            }
            __syncthreads();
        }

        // =============== Y: this CTA's row pairs, a warp takes NPW of them at a time, __syncwarp only ===============
        {
            const int lane = opaque(lane0);
            const int k1y = lane < AY ? lane : lane - AY;   // lanes >= AY shadow an item (same addresses) and skip the stores
            const bool act2 = lane < AY;
            const int j1 = (lane / BY) < NPW ? (lane / BY) : 0;   // Y1 / Y3 item: pair j1 of the warp item, position lane mod BY
            const bool act1 = (lane / BY) < NPW;
            const int n2 = lane % BY;
            constexpr bool TWREG = (BY == 8);                     // the lane's y twiddles in registers (else read at every use)
            cplx* Zw = A + (warp * NF * NPW) * PS;                // this warp's pair storages: g, then (CHIV) chi
            [[maybe_unused]] cplx tq[BY];
            if constexpr (TWREG) {
#pragma unroll
                for (int k2 = 1; k2 < BY; ++k2) tq[k2] = twy[k1y * BYP + k2];
            }
            // Y1: pruned radix-AY of rows m (h = 0: second half of the storage) / m + NX/2 (h = 1: first half) of the NPW
            // pairs that start at storage Zst; the exchange tile of a pair starts at its row m
            auto y1 = [&](cplx* Zst, int h) {
                const cplx* Zr = Zst + j1 * PS + (h ? 0 : W2) + n2;
                cplx lo[AY1], hi[AY1];
#pragma unroll
                for (int a = 0; a < AY1; ++a) {
                    lo[a] = Zr[BY * a];
                    hi[a] = Zr[BY * a + NKY0];
                }
                cplx out[AY];
                dft_pruned_in<AY, +1>(lo, hi, out);
                __syncwarp(FULL);  // h = 0: rows m are in registers before the tiles overwrite them; h = 1: Y2 done
                if (act1) {
                    cplx* tile = Zst + j1 * PS + W2 + n2;
#pragma unroll
                    for (int k1 = 0; k1 < AY; ++k1) tile[k1 * BYP] = out[k1];
                }
            };
            // (dx chi, dy chi) of row `row` at y = k1 + AY k2, k2 < 8, from the real-space rows (EM: composed from two fields)
            auto load_chi = [&](cplx (&c)[BY], int row, int k1) {
                const size_t off = (size_t)row * NY + k1;
#pragma unroll
                for (int k2 = 0; k2 < BY; ++k2) c[k2] = ldg_nc_early(Rc + off + AY * k2);
                if constexpr (EM) {
#pragma unroll
                    for (int k2 = 0; k2 < BY; ++k2) {
                        const cplx a2 = ldg_nc_early(Rc2 + off + AY * k2);
                        c[k2] = cmake(fma(-vpar, a2.x, c[k2].x), fma(-vpar, a2.y, c[k2].y));
                    }
                }
            };
#pragma unroll 1
            for (int item = warp; item < K::NITEM; item += NW) {
                const int q0 = rank * PPG + item * NPW;           // first pair of the item
                if (lane == 0) {   // the rows of the item's pairs: one bulk copy per pair and field (2 W2 values, contiguous in Z)
                    // generic-proxy accesses before, async-proxy copies after: the scratch rows other SMs wrote (first item
                    // after the hand-over: the full fence) and this warp's tiles, which the copies overwrite (every item: the
                    // shared-memory fence is enough; measured 1-2 % of the kernel)
                    if (item == warp) fence_proxy_async(); else fence_proxy_async_smem();
                    mbar_arrive_expect_tx(ybar, (uint32_t)(NF * NPW * 2 * W2 * sizeof(cplx)));
#pragma unroll
                    for (int j = 0; j < NF * NPW; ++j)
                        bulk_g2s_hint(smem_u32(Zw + j * PS), Zs + (size_t)(j / NPW) * K::ZS_CPLX + (size_t)(q0 + j % NPW) * (2 * W2),
                                      (uint32_t)(2 * W2 * sizeof(cplx)), ybar, pol_keep);
                }
                [[maybe_unused]] cplx chv[BY];
                if constexpr (!CHIV && !(((NPW * AY + 31) / 32) < NPW)) load_chi(chv, q0, k1y);   // (flat items: below)
                mbar_wait(ybar, yph);
                yph ^= 1;
                // The rows are in shared memory: their lines in the scratch are dead.  Dropping them pays where the groups'
                // scratch exceeds what L2 keeps (768 x 384: 85 MB; DRAM writes 69 -> 34 GB per launch, time unchanged;
                // 144 x 144 with 148 groups of one CTA: 82 MB; DRAM traffic 2.0 -> 1.05 x the algorithmic bytes for 2 % of
                // the time); at 384 x 192 (44 MB, already 1.05 x) it cost 14 % of the time: not done there.
                if constexpr (K::DISCARD) {
                    constexpr int LPB = (int)(2 * W2 * sizeof(cplx) / 128);   // lines per pair block
                    for (int i = lane; i < NF * NPW * LPB; i += 32) {
                        const int j = i / LPB;
                        l2_discard_line(Zs + (size_t)(j / NPW) * K::ZS_CPLX + (size_t)(q0 + j % NPW) * (2 * W2) + (size_t)(i % LPB) * 8);
                    }
                }
                // Y2 items (pair j, k1): NPW AY of them.  With AY lanes per pair a round is one pair (AY of 32 lanes busy);
                // when fewer rounds of 32 cover all items (AY = 18: 54 items, 2 rounds instead of 3) the items are laid
                // flat over the lanes and the twiddles of a lane's k1 are read again for every round.
                constexpr int NY2 = NPW * AY, NRF = (NY2 + 31) / 32;
                constexpr bool FLAT = NRF < NPW;
                constexpr int NR = FLAT ? NRF : NPW;
                constexpr bool AHEAD = (BY == 8);                     // chi values of the next round in a second register set
                double nlx[NR][BY];                                   // bracket of the rows m (first halves), kept in registers
                auto item_of = [&](int r, int& j, int& k1, bool& valid) {
                    if constexpr (FLAT) {
                        const int idx = r * 32 + lane;
                        valid = idx < NY2;
                        const int ic = valid ? idx : idx - 32;       // idle lanes shadow an item of the previous round
                        j = ic / AY;
                        k1 = ic % AY;
                    } else {
                        j = r;
                        k1 = k1y;
                        valid = act2;
                    }
                };
                if constexpr (FLAT && !CHIV) {   // the first round's chi values for the flat item of this lane
                    int j, k1; bool valid;
                    item_of(0, j, k1, valid);
                    load_chi(chv, q0 + j, k1);
                }
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    y1(Zw, h);
                    if constexpr (CHIV) y1(Zw + NPW * PS, h);
                    __syncwarp(FULL);
#pragma unroll
                    for (int r = 0; r < NR; ++r) {  // Y2: twiddle + radix-8 to real space, bracket
                        int j, k1; bool valid;
                        item_of(r, j, k1, valid);
                        // chi values of the NEXT round (or of the first round of the second half): requested before this
                        // round's butterflies (AHEAD: into a second register set) or right after this round's bracket
                        auto next_chi = [&](cplx (&dst)[BY]) {
                            const int rn = (r + 1 < NR) ? r + 1 : 0, hn = (r + 1 < NR) ? h : 1;
                            if (!(h == 1 && r + 1 == NR)) {
                                int jn, k1n; bool vn;
                                item_of(rn, jn, k1n, vn);
                                load_chi(dst, q0 + jn + hn * NPAIR, k1n);
                            }
                        };
                        [[maybe_unused]] cplx chn[AHEAD ? BY : 1];
                        if constexpr (!CHIV && AHEAD) next_chi(chn);
                        const cplx* twl = twy + k1 * BYP;   // the item's twiddles W_NY^{k1 k2} (when they are not in registers)
                        [[maybe_unused]] cplx tqr[8];
                        if constexpr (FLAT && BY == 8) {
#pragma unroll
                            for (int k2 = 1; k2 < 8; ++k2) tqr[k2] = twl[k2];
                        }
                        // twiddle + radix-BY to real space
                        auto to_real = [&](cplx (&x)[BY]) {
                            if constexpr (BY == 8) {
                                if constexpr (FLAT) dft8_twiddled<+1>(x, tqr); else dft8_twiddled<+1>(x, tq);
                            } else {
#pragma unroll
                                for (int i = 1; i < BY; ++i) { const cplx w = twl[i]; x[i] = cmul(x[i], w.x, w.y); }
                                Dft<BY, +1>::run(x);
                            }
                        };
                        cplx* tile = Zw + j * PS + W2 + k1 * BYP;
                        cplx v[BY];
#pragma unroll
                        for (int i = 0; i < BY; ++i) v[i] = tile[i];
                        to_real(v);                 // (dx g + i dy g)(row, y = k1 + AY k2)
                        if constexpr (CHIV) {       // (dx chi + i dy chi) of the same row from chi's tile
                            const cplx* tc = Zw + (NPW + j) * PS + W2 + k1 * BYP;
#pragma unroll
                            for (int i = 0; i < BY; ++i) chv[i] = tc[i];
                            to_real(chv);
                        }
                        if (h == 0) {
#pragma unroll
                            for (int k2 = 0; k2 < BY; ++k2) nlx[r][k2] = fma(chv[k2].x, v[k2].y, -chv[k2].y * v[k2].x);
                            if constexpr (!CHIV && !AHEAD) next_chi(chv);
                        } else {
                            cplx w[BY];
#pragma unroll
                            for (int k2 = 0; k2 < BY; ++k2)
                                w[k2] = cmake(nlx[r][k2], fma(chv[k2].x, v[k2].y, -chv[k2].y * v[k2].x));
                            if constexpr (!CHIV && !AHEAD) next_chi(chv);
                            Dft<BY, -1>::run(w);
#pragma unroll
                            for (int k2 = 1; k2 < BY; ++k2) {
                                cplx t;
                                if constexpr (BY == 8) t = FLAT ? tqr[k2] : tq[k2]; else t = twl[k2];
                                w[k2] = cmul(w[k2], t.x, -t.y);
                            }
                            if (valid) {  // own slots of the tile: no other active lane reads or writes them in this phase
#pragma unroll
                                for (int k2 = 0; k2 < BY; ++k2) tile[k2] = w[k2];
                            }
                        }
                        if constexpr (!CHIV && AHEAD) {
                            if (!(h == 1 && r + 1 == NR)) {
#pragma unroll
                                for (int k2 = 0; k2 < BY; ++k2) chv[k2] = chn[k2];
                            }
                        }
                    }
                    __syncwarp(FULL);
                }
                {  // Y3: pruned-output radix-AY; P[pair][cc] goes to global memory (L2), 128 B runs
                    const cplx* tile = Zw + j1 * PS + W2 + n2;
                    cplx in[AY];
#pragma unroll
                    for (int n1 = 0; n1 < AY; ++n1) in[n1] = tile[n1 * BYP];
                    cplx lo[AY1], hi[AY1];
                    dft_pruned_out<AY, -1>(in, lo, hi);
                    if (act1) {
                        cplx* Pp = Ps + (size_t)(q0 + j1) * W2 + n2;
#pragma unroll
                        for (int c = 0; c < AY1; ++c) {
                            stg_hint(Pp + BY * c, lo[c], pol_keep);          // +ky half: cc = ky = n2 + BY c
                            stg_hint(Pp + BY * c + NKY0, hi[c], pol_keep);   // -ky half: cc = nky0 + n2 + BY c  <->  ky = nky0 - n2 - BY c
                        }
                    }
                }
                __syncwarp(FULL);   // the tiles are consumed before the next item's rows land on them
            }
        }
        // ---- hand-over 2: every CTA of the group has written its rows of P ----
        __syncthreads();
        if constexpr (G > 1) {
            if (tid == 0) {
                __threadfence();
                atomicAdd(pcnt, 1u);
                while (ld_acquire_gpu(pcnt) < (unsigned)G * (it + 1)) {}
            }
            __syncthreads();
        }

        // =============== X2: x-analysis of this CTA's column units, UPP at a time; delete modes, prefactor, add ===============
        if (tid == 0 && t + (unsigned)ngroup < T) request_block(t + (unsigned)ngroup, 0);   // lands behind the x tiles
        {
            cplx r0[AX21], r1[AX21];
            const int k2s = tid % BX2, cols = (tid / BX2) % CK, us = tid / (BX2 * CK);   // stage 2 item: (unit us of the pass, column, k2)
            const bool has2 = tid < UPP * CK * BX2;
#pragma unroll 1
            for (int ub = 0; ub < UPC; ub += UPP) {
#pragma unroll 1
                for (int i1 = tid; i1 < UPP * CK * AX2; i1 += NT) {
                    // stage 1: unpack the row pair, radix-BX2 over n2 for fixed n1 (m = n1 + AX2 n2), twiddle
                    const int col = i1 % CK, n1 = (i1 / CK) % AX2, ul = i1 / (CK * AX2);
                    const int kyi = (rank + G * (ub + ul)) * CK + col;
                    const int ccm = kyi ? W2 - kyi : 0;
                    cplx x[BX2];
#pragma unroll
                    for (int i = 0; i < C22; ++i) {
                        const cplx* Pr = Ps + (size_t)(n1 + AX2 * i) * W2;
                        const cplx pp = ldg_cg_hint(Pr + kyi, pol_keep), pm = ldg_cg_hint(Pr + ccm, pol_keep);
                        x[i] = cmake(pp.x + pm.x, pp.y - pm.y);          // 2 N^_m  = P+ + conj P-
                        x[i + C22] = cmake(pp.y + pm.y, pm.x - pp.x);    // 2 N^_m' = -i (P+ - conj P-)
                    }
                    Dft<BX2, -1>::run(x);
                    cplx* Ec = A + (ul * CK + col) * CSF + n1 * BPX2;
#pragma unroll
                    for (int k2 = 0; k2 < BX2; ++k2) {
                        const cplx w = twx2[n1 * BPX2 + k2];
                        Ec[k2] = (k2 == 0) ? x[0] : cmul(x[k2], w.x, -w.y);
                    }
                    // the +ky halves of these P rows (one 128-byte line per row and unit, read by this warp instruction only)
                    // are dead: drop them from L2 where the groups' scratch exceeds what L2 keeps
                    if constexpr (K::DISCARD && CK == 8) {
                        // the other seven lanes of the line have their values too before it is dropped (whole warps run
                        // this loop, so the warp barrier is met by all 32 lanes)
                        static_assert((UPP * CK * AX2) % 32 == 0, "whole warps in the stage-1 loop of X2");
                        __syncwarp(FULL);
                        if (col == 0) {
#pragma unroll
                            for (int i = 0; i < C22; ++i) l2_discard_line(Ps + (size_t)(n1 + AX2 * i) * W2 + kyi);
                        }
                    }
                }
                cplx* Rcol = Rb + (size_t)((rank + G * (ub + us)) * CK + cols) * NX0 + k2s;
                if (has2) {  // rhs values of this thread's share of stage 2
#pragma unroll
                    for (int c = 0; c < AX21; ++c) {
                        r0[c] = ldg_early(Rcol + BX2 * c);
                        r1[c] = ldg_early(Rcol + BX2 * c + M);
                    }
                }
                __syncthreads();
                if (has2) {  // stage 2: pruned-output radix-AX2 over n1 for fixed k2; i = k2 + BX2 c
                    cplx in[AX2];
                    const cplx* Ec = A + (us * CK + cols) * CSF + k2s;
#pragma unroll
                    for (int n1 = 0; n1 < AX2; ++n1) in[n1] = Ec[n1 * BPX2];
                    cplx lo[AX21], hi[AX21];
                    dft_pruned_out<AX2, -1>(in, lo, hi);
#pragma unroll
                    for (int c = 0; c < AX21; ++c) {
                        Rcol[BX2 * c] = cmake(fma(coef, lo[c].x, r0[c].x), fma(coef, lo[c].y, r0[c].y));
                        if (c != 0 || k2s != 0)  // i = M is the Nyquist row: untouched (R6)
                            Rcol[BX2 * c + M] = cmake(fma(coef, hi[c].x, r1[c].x), fma(coef, hi[c].y, r1[c].y));
                    }
                }
                __syncthreads();  // the tiles are consumed before the next pass / the next plane's E overwrites them
            }
        }
    }
}

}  // namespace gnl
