// nl_wa.cuh -- the fused per-plane kernel for planes beyond one SM, WARP-AUTONOMOUS: the group kernel of nl_group.cuh
// (a plane spread over a group of G co-resident CTAs, x<->y hand-overs through a per-group scratch that lives in L2)
// with no CTA-wide barrier left in the plane loop.
//
// Same steps and the same scratch layout as nl_group.cuh.  What the ncu capture of
// that kernel showed (profiles/r02_ncu_summary.md): its y phase -- warps that run whole row pairs with
// __syncwarp only -- issues 54 % of the instructions in 36 % of the time, while the two x phases, whose 8 warps move
// in lockstep through stage 1 / __syncthreads / stage 2 / __syncthreads, need 60 % of the time for the rest: in
// lockstep all warps load, then all compute, then all store, so the FP64 pipe idles while the shared-memory pipe works
// and vice versa.  Here the x phases are warp tasks as well:
//   X1  a warp takes CW = 2 ADJACENT stored columns through both x stages (pruned radix-AX, twiddle, exchange through
//       its own shared-memory tile, radix-BX) and stores the rows to Z from registers; adjacent columns make every
//       store a full 32-byte sector.  The +ky columns are paired (2u, 2u+1), the -ky columns (2u+1, 2u+2), so that
//       their slots cc = W2 - ky pair up sector-aligned too (ky = nky0 is the all-zero slot cc = nky0).
//   Y   as in nl_group.cuh: a warp takes NPW row pairs at a time; rows come in by 1-D bulk copies (TMA).
//   X2  a warp takes 2 adjacent columns: unpack the row pairs of P, radix-BX2, twiddle, exchange, pruned-output
//       radix-AX2, delete modes, prefactor, rhs +=.
// A warp owns one slice of shared memory that serves its tasks in turn (x tile / pair storages), so warps never wait
// for one another inside a CTA; the two hand-overs of a plane are counters per group that every WARP arrives on
// (__syncwarp, __threadfence + atomicAdd by lane 0) and polls.  Warps drift apart and the FP64 work of one overlaps
// the shared-memory and L2 traffic of the others, in every phase.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "nl_group.cuh"

namespace gnl {

__host__ __device__ constexpr int pad_4mod8(int n) { return n + ((4 - n % 8) + 8) % 8; }
__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }

// Nx = AX * BX (x-synthesis) = AX2 * BX2 (x-analysis), Ny = AY * BY; G CTAs of NW warps per group; NPW row pairs per
// y item; CHIV: chi per plane goes through X1 and the row hand-over like g.
template <int AX_, int BX_, int AY_, int BY_, int G_, int NW_, bool CHIV_, int NPW_, int AX2_ = 0, int BX2_ = 0>
struct WarpAuto {
    static constexpr int AX = AX_, BX = BX_, AY = AY_, BY = BY_, BYP = BY_ + 1, G = G_, NW = NW_, NPW = NPW_;
    static constexpr int AX2 = AX2_ ? AX2_ : AX_, BX2 = BX2_ ? BX2_ : BX_;
    static constexpr bool CHIV = CHIV_;
    static constexpr int NF = CHIV ? 2 : 1;
    static constexpr int NX = AX * BX, NY = AY * BY, NKY0 = NY / 3, W2 = 2 * NKY0, NPAIR = NX / 2, M = NX / 3, NX0 = 2 * M;
    static constexpr int C2 = BX / 2, C22 = BX2 / 2;
    static constexpr int CW = 2;                       // adjacent stored columns per x task
    static constexpr int NXT = NKY0 / CW;              // x tasks per plane and field
    static constexpr int GW = G * NW;                  // warps of a group
    static constexpr int PPG = NPAIR / G, NITEM = PPG / NPW;
    static constexpr int NT = 32 * NW;
    static constexpr int BPX = Tile<AX, BX>::BP, BPX2 = Tile<AX2, BX2>::BP;
    // x tile of one column [k1][BPX]; column stride = 4 mod 8 keeps the lanes (column, k1) of stage 2 conflict free
    static constexpr int TJ1 = pad_4mod8(AX * BPX), TJ2 = pad_4mod8(AX2 * BPX2);
    static constexpr int FY = AY * BYP, PS = (W2 + FY) | 1;
    static constexpr int SLICE = cmax(NF * NPW * PS, cmax(CW * TJ1, CW * TJ2)) + (cmax(NF * NPW * PS, cmax(CW * TJ1, CW * TJ2)) & 1);
    static constexpr int TWX = AX * BPX, TWY = AY * BYP;
    static constexpr int TWX2 = (AX2 == AX && BX2 == BX) ? 0 : AX2 * BPX2;
    static constexpr int SMEM_CPLX = NW * SLICE + TWX + TWX2 + TWY + (NW + 1) / 2;
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)SMEM_CPLX;
    static constexpr size_t ZS_CPLX = (size_t)NPAIR * 2 * W2, PS_CPLX = (size_t)NPAIR * W2;   // per-group scratch
    static constexpr size_t GROUP_SCRATCH_CPLX = NF * ZS_CPLX + PS_CPLX;
    static_assert(AX % 3 == 0 && AY % 3 == 0 && AX2 % 3 == 0 && BX % 2 == 0 && BX2 % 2 == 0, "3/2 rule; row pairs");
    static_assert(AX2 * BX2 == NX && NKY0 % CW == 0 && NPAIR % G == 0 && PPG % NPW == 0, "the group divides the work");
    static_assert(NPW * BY <= 32 && AY <= 32 && NKY0 == BY * (AY / 3) && (BY == 8 || BY == 16), "lanes of the y stages");
};

// One warp of every group arrives on a hand-over counter and waits until all GW warps of the group have arrived `round`
// times (counters are monotonic over the launch).
__device__ __forceinline__ void wa_handover(unsigned* cnt, unsigned target, int lane)
{
    __syncwarp(0xffffffffu);
    if (lane == 0) {
        __threadfence();
        atomicAdd(cnt, 1u);
    }
    // every lane polls (one request per warp: same address) and the exit test is made warp-uniform: with the spin loop
    // inside the lane-0 branch the warp was measured to stay split (lane 0 | the other 31) for the rest of the kernel
    while (__shfl_sync(0xffffffffu, ld_acquire_gpu(cnt), 0) < target) __nanosleep(32);
    __syncwarp(0xffffffffu);
}

// A round of 32 lanes over NITEMS items: lanes beyond the last item SHADOW an item of their own (same addresses: the
// shared-memory loads broadcast) and only skip the stores, so that a task has no divergent region -- a warp that splits
// at a half-warp condition here was measured to stay split for the rest of the kernel (every instruction issued twice).
template <int NITEMS>
__device__ __forceinline__ int wa_item(int r, int lane, bool& valid)
{
    const int i = 32 * r + lane;
    if constexpr (NITEMS % 32 == 0) {
        valid = true;
        return i;
    } else {
        valid = i < NITEMS;
        return valid ? i : i % (NITEMS % 32 < 32 ? NITEMS % 32 : 32);   // an item of the last (partial) round's first lanes
    }
}

// ---- X1 task: the x-synthesis of two adjacent columns of one sign; rows go to Zf from registers --------------------
// sg = 0: columns ky = kyA, kyA + 1 (+ky: (i kx - ky) F -> slot cc = ky); sg = 1: columns ky = kyA + 1, kyA + 2 stored
// conjugated in slots cc = W2 - ky (ky = nky0: the all-zero slot cc = nky0).  kyA is even.
// Stage-1 item of round r: (column j, position n2).  x1_load requests the item's non-zero inputs (i = n2 + BX a and
// n2 + BX a + M); x1_stage1 runs derivative, pad, pruned radix-AX over n1 and the twiddle W_NX^{n2 k1} into the tile.
template <class K>
__device__ __forceinline__ void x1_load(const cplx* __restrict__ F, int kyA, int sg, int r, int lane, cplx (&lo)[K::AX / 3],
                                        cplx (&hi)[K::AX / 3])
{
    constexpr int AX1 = K::AX / 3, BX = K::BX, M = K::M, NX0 = K::NX0, NKY0 = K::NKY0, CW = K::CW;
    bool valid;
    const int i = wa_item<CW * BX>(r, lane, valid);
    const int j = i / BX, n2 = i % BX;
    const int kyi = kyA + sg + j;
    const int kyc = kyi < NKY0 ? kyi : NKY0 - 1;   // ky = nky0: there is no such column (x1_stage1 makes it zero)
    const cplx* Fc = F + (size_t)kyc * NX0 + n2;
#pragma unroll
    for (int a = 0; a < AX1; ++a) {
        lo[a] = ldg_nc_early(Fc + BX * a);
        hi[a] = ldg_nc_early(Fc + BX * a + M);
    }
    if (kyA + sg == 0) {  // (warp-uniform) the task holds the ky = 0 column: its Hermitian part is used (reading R7)
#pragma unroll
        for (int a = 0; a < AX1; ++a) {
            const int i0 = n2 + BX * a, i1 = i0 + M;
            const cplx m0 = F[(size_t)kyc * NX0 + (NX0 - i0) % NX0], m1 = F[(size_t)kyc * NX0 + NX0 - i1];
            if (j == 0) {
                lo[a] = cmake(0.5 * (lo[a].x + m0.x), 0.5 * (lo[a].y - m0.y));
                hi[a] = cmake(0.5 * (hi[a].x + m1.x), 0.5 * (hi[a].y - m1.y));
            }
        }
    }
}
template <class K>
__device__ __forceinline__ void x1_stage1(cplx (&lo)[K::AX / 3], cplx (&hi)[K::AX / 3], cplx* E, const cplx* twx, int kyA, int sg,
                                          int r, int lane, double kxmin, double kymin)
{
    constexpr int AX = K::AX, BX = K::BX, AX1 = AX / 3, BPX = K::BPX, TJ = K::TJ1, CW = K::CW;
    constexpr int M = K::M, NX0 = K::NX0, NKY0 = K::NKY0;
    bool valid;
    const int i = wa_item<CW * BX>(r, lane, valid);
    const int j = i / BX, n2 = i % BX;
    const int kyi = kyA + sg + j;
    const double zf = kyi < NKY0 ? 1.0 : 0.0;   // ky = nky0: slot cc = nky0 holds zeros (a zero factor makes them exact)
    const double ky = zf * kymin * (double)kyi, dn2 = (double)n2, kxs = zf * kxmin;
    const double kys = sg ? ky : -ky;           // (i kx - ky) F for +ky, (i kx + ky) F for -ky
#pragma unroll
    for (int a = 0; a < AX1; ++a) {
        lo[a] = deriv_mul(lo[a], kxs * (dn2 + (double)(BX * a)), kys);                // i = n2 + BX a      (kx >= 0)
        hi[a] = deriv_mul(hi[a], kxs * (dn2 + (double)(BX * a + M - NX0)), kys);      // i = n2 + BX a + M  (kx < 0)
    }
    if (n2 == 0) hi[0] = cmake(0.0, 0.0);  // i = M: the Nyquist row is ignored (R6)
    cplx out[AX];
    dft_pruned_in<AX, +1>(lo, hi, out);
    cplx* Ec = E + j * TJ + n2;
    const cplx* tw = twx + n2;
    if (valid) Ec[0] = out[0];
#pragma unroll
    for (int k1 = 1; k1 < AX; ++k1) {
        const cplx w = tw[k1 * BPX];
        const cplx o = cmul(out[k1], w.x, w.y);
        if (valid) Ec[k1 * BPX] = o;
    }
}
// stage 2: item (column j, k1): radix-BX over n2; row m = k1 + AX k2 is half k2 / C2 of pair k1 + AX (k2 mod C2)
template <class K>
__device__ __forceinline__ void x1_stage2(const cplx* E, cplx* __restrict__ Zf, int kyA, int sg, int lane, uint64_t pol_keep)
{
    constexpr int AX = K::AX, BX = K::BX, BPX = K::BPX, TJ = K::TJ1, CW = K::CW, C2 = K::C2, W2 = K::W2;
    constexpr int R2 = (CW * AX + 31) / 32;
#pragma unroll
    for (int r = 0; r < R2; ++r) {
        bool valid;
        const int i = wa_item<CW * AX>(r, lane, valid);
        const int j = i % CW, k1 = i / CW;
        const int kyi = kyA + sg + j;
        cplx v[BX];
        const cplx* Ec = E + j * TJ + k1 * BPX;
#pragma unroll
        for (int n2 = 0; n2 < BX; ++n2) v[n2] = Ec[n2];
        Dft<BX, +1>::run(v);
        const int cc = sg ? W2 - kyi : kyi;
        cplx* Zc = Zf + (size_t)k1 * (2 * W2) + cc;
        const double sgn = sg ? -1.0 : 1.0;   // -ky columns hold the conjugate
#pragma unroll
        for (int k2 = 0; k2 < BX; ++k2) {     // pair storage: row m + NX/2 (k2 >= C2) first, then row m
            if (valid) stg_hint(Zc + (size_t)(AX * (k2 % C2)) * (2 * W2) + (k2 < C2 ? W2 : 0), cmake(v[k2].x, sgn * v[k2].y), pol_keep);
        }
    }
}
// PF: the inputs of the second sign are requested before the second stage of the first one (one stage-1 round only)
template <class K, bool PF>
__device__ __forceinline__ void wa_x1_task(const cplx* __restrict__ F, cplx* __restrict__ Zf, cplx* E, const cplx* twx, int kyA,
                                           int lane, double kxmin, double kymin, uint64_t pol_keep)
{
    constexpr int AX1 = K::AX / 3, R1 = (K::CW * K::BX + 31) / 32;
    constexpr unsigned FULL = 0xffffffffu;
    if constexpr (PF && R1 == 1) {
        cplx lo[AX1], hi[AX1];
        x1_load<K>(F, kyA, 0, 0, lane, lo, hi);
        x1_stage1<K>(lo, hi, E, twx, kyA, 0, 0, lane, kxmin, kymin);
        __syncwarp(FULL);
        x1_load<K>(F, kyA, 1, 0, lane, lo, hi);
        x1_stage2<K>(E, Zf, kyA, 0, lane, pol_keep);
        __syncwarp(FULL);   // the tile is consumed before the next sign overwrites it
        x1_stage1<K>(lo, hi, E, twx, kyA, 1, 0, lane, kxmin, kymin);
        __syncwarp(FULL);
        x1_stage2<K>(E, Zf, kyA, 1, lane, pol_keep);
        __syncwarp(FULL);
    } else {
#pragma unroll 1
        for (int sg = 0; sg < 2; ++sg) {
#pragma unroll
            for (int r = 0; r < R1; ++r) {
                cplx lo[AX1], hi[AX1];
                x1_load<K>(F, kyA, sg, r, lane, lo, hi);
                x1_stage1<K>(lo, hi, E, twx, kyA, sg, r, lane, kxmin, kymin);
            }
            __syncwarp(FULL);
            x1_stage2<K>(E, Zf, kyA, sg, lane, pol_keep);
            __syncwarp(FULL);   // the tile is consumed before the next sign / task overwrites it
        }
    }
}

// ---- X2 task: the x-analysis of two adjacent columns ky = kyA, kyA + 1; delete modes, prefactor, rhs += ------------
// stage 1: item (column j, n1): unpack the row pairs, radix-BX2 over n2 (m = n1 + AX2 n2), twiddle W_NX^{-n1 k2}
template <class K>
__device__ __forceinline__ void x2_load_p(const cplx* __restrict__ Ps, int kyA, int r, int lane, cplx (&pp)[K::BX2 / 2],
                                          cplx (&pm)[K::BX2 / 2], uint64_t pol_keep)
{
    constexpr int AX2 = K::AX2, CW = K::CW, C22 = K::C22, W2 = K::W2;
    bool valid;
    const int i = wa_item<CW * AX2>(r, lane, valid);
    const int j = i % CW, n1 = i / CW;
    const int kyi = kyA + j;
    const int ccm = kyi ? W2 - kyi : 0;
#pragma unroll
    for (int ii = 0; ii < C22; ++ii) {
        const cplx* Pr = Ps + (size_t)(n1 + AX2 * ii) * W2;
        pp[ii] = ldg_cg_hint(Pr + kyi, pol_keep);
        pm[ii] = ldg_cg_hint(Pr + ccm, pol_keep);
    }
}
template <class K>
__device__ __forceinline__ void x2_stage1(const cplx (&pp)[K::BX2 / 2], const cplx (&pm)[K::BX2 / 2], cplx* E, const cplx* twx2,
                                          int r, int lane)
{
    constexpr int AX2 = K::AX2, BX2 = K::BX2, BPX2 = K::BPX2, TJ = K::TJ2, CW = K::CW, C22 = K::C22;
    bool valid;
    const int i = wa_item<CW * AX2>(r, lane, valid);
    const int j = i % CW, n1 = i / CW;
    cplx x[BX2];
#pragma unroll
    for (int ii = 0; ii < C22; ++ii) {
        x[ii] = cmake(pp[ii].x + pm[ii].x, pp[ii].y - pm[ii].y);          // 2 N^_m  = P+ + conj P-
        x[ii + C22] = cmake(pp[ii].y + pm[ii].y, pm[ii].x - pp[ii].x);    // 2 N^_m' = -i (P+ - conj P-)
    }
    Dft<BX2, -1>::run(x);
    cplx* Ec = E + j * TJ + n1 * BPX2;
    const cplx* tw = twx2 + n1 * BPX2;
    if (valid) Ec[0] = x[0];
#pragma unroll
    for (int k2 = 1; k2 < BX2; ++k2) {
        const cplx w = tw[k2];
        const cplx o = cmul(x[k2], w.x, -w.y);
        if (valid) Ec[k2] = o;
    }
}
// stage 2: item (column j, k2): pruned-output radix-AX2 over n1; i = k2 + BX2 c
template <class K>
__device__ __forceinline__ void x2_load_r(cplx* __restrict__ Rb, int kyA, int r, int lane, cplx (&r0)[K::AX2 / 3], cplx (&r1)[K::AX2 / 3])
{
    constexpr int AX21 = K::AX2 / 3, BX2 = K::BX2, CW = K::CW, M = K::M, NX0 = K::NX0;
    bool valid;
    const int i = wa_item<CW * BX2>(r, lane, valid);
    const cplx* Rcol = Rb + (size_t)(kyA + i % CW) * NX0 + i / CW;
#pragma unroll
    for (int c = 0; c < AX21; ++c) {
        r0[c] = ldg_early(Rcol + BX2 * c);
        r1[c] = ldg_early(Rcol + BX2 * c + M);
    }
}
template <class K>
__device__ __forceinline__ void x2_stage2(const cplx* E, cplx* __restrict__ Rb, int kyA, int r, int lane, const cplx (&r0)[K::AX2 / 3],
                                          const cplx (&r1)[K::AX2 / 3], double coef)
{
    constexpr int AX2 = K::AX2, BX2 = K::BX2, AX21 = AX2 / 3, BPX2 = K::BPX2, TJ = K::TJ2, CW = K::CW, M = K::M, NX0 = K::NX0;
    bool valid;
    const int i = wa_item<CW * BX2>(r, lane, valid);
    const int j = i % CW, k2 = i / CW;
    cplx* Rcol = Rb + (size_t)(kyA + j) * NX0 + k2;
    cplx in[AX2];
    const cplx* Ec = E + j * TJ + k2;
#pragma unroll
    for (int n1 = 0; n1 < AX2; ++n1) in[n1] = Ec[n1 * BPX2];
    cplx lo[AX21], hi[AX21];
    dft_pruned_out<AX2, -1>(in, lo, hi);
#pragma unroll
    for (int c = 0; c < AX21; ++c) {
        if (valid) Rcol[BX2 * c] = cmake(fma(coef, lo[c].x, r0[c].x), fma(coef, lo[c].y, r0[c].y));
        if (valid && (c != 0 || k2 != 0))  // i = M is the Nyquist row: untouched (R6)
            Rcol[BX2 * c + M] = cmake(fma(coef, hi[c].x, r1[c].x), fma(coef, hi[c].y, r1[c].y));
    }
}
// PF: every round's P values are requested before the first round's butterflies, the rhs values of the first stage-2
// round before the last stage-1 round's butterflies
template <class K, bool PF>
__device__ __forceinline__ void wa_x2_task(const cplx* __restrict__ Ps, cplx* __restrict__ Rb, cplx* E, const cplx* twx2, int kyA,
                                           int lane, double coef, uint64_t pol_keep)
{
    constexpr int C22 = K::C22, AX21 = K::AX2 / 3;
    constexpr int R1 = (K::CW * K::AX2 + 31) / 32, R2 = (K::CW * K::BX2 + 31) / 32;
    constexpr unsigned FULL = 0xffffffffu;
    cplx r0[AX21], r1[AX21];
    if constexpr (PF && R1 <= 2) {
        cplx pp[R1][C22], pm[R1][C22];
#pragma unroll
        for (int r = 0; r < R1; ++r) x2_load_p<K>(Ps, kyA, r, lane, pp[r], pm[r], pol_keep);
#pragma unroll
        for (int r = 0; r < R1; ++r) {
            if (r == R1 - 1) x2_load_r<K>(Rb, kyA, 0, lane, r0, r1);
            x2_stage1<K>(pp[r], pm[r], E, twx2, r, lane);
        }
    } else {
#pragma unroll
        for (int r = 0; r < R1; ++r) {
            cplx pp[C22], pm[C22];
            x2_load_p<K>(Ps, kyA, r, lane, pp, pm, pol_keep);
            x2_stage1<K>(pp, pm, E, twx2, r, lane);
        }
    }
    __syncwarp(FULL);
#pragma unroll
    for (int r = 0; r < R2; ++r) {
        if (!(PF && R1 <= 2) || r > 0) x2_load_r<K>(Rb, kyA, r, lane, r0, r1);
        x2_stage2<K>(E, Rb, kyA, r, lane, r0, r1, coef);
    }
    __syncwarp(FULL);   // the tile is consumed before the next task overwrites it
}

// [first, first + bytes) towards L2 with ONE bulk-prefetch instruction (TMA; bytes a multiple of 16).  A loop of
// prefetch.global.L2 per 128-byte line was measured at 10 % of the kernel's stall samples (the LSU queue throttles).
__device__ __forceinline__ void wa_prefetch(const void* first, size_t bytes, int lane)
{
    if (lane == 0) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(first), "r"((uint32_t)bytes) : "memory");
}

// grid = groups * G CTAs (cooperative launch: every CTA is resident).  Arguments as k_plane_group; cnt: 2 * groups
// counters, zeroed before the launch.
template <int AX, int BX, int AY, int BY, int G, int NW, bool CHIV, bool EM, int NPW_, bool PF, int AX2_ = 0, int BX2_ = 0>
__global__ void __launch_bounds__(32 * NW, 1)
k_plane_wa(const cplx* __restrict__ g, cplx* __restrict__ rhs, const cplx* __restrict__ R, const cplx* __restrict__ chi,
           const cplx* __restrict__ twx_g, const cplx* __restrict__ twy_g, cplx* __restrict__ scratch,
           unsigned* __restrict__ cnt, int nz, int nv, int nslab, double kxmin, double kymin, double coef,
           const cplx* __restrict__ R2 = nullptr, const double* __restrict__ vp = nullptr, int nw = 1, int slab0 = 0)
{
    static_assert(!(EM && CHIV), "the composition needs chi-like fields shared over v");
    using K = WarpAuto<AX, BX, AY, BY, G, NW, CHIV, NPW_, AX2_, BX2_>;
    constexpr int BYP = K::BYP, NX = K::NX, NY = K::NY, NKY0 = K::NKY0, W2 = K::W2, NPAIR = K::NPAIR, NF = K::NF;
    constexpr int NX0 = K::NX0, PPG = K::PPG, NPW = K::NPW, PS = K::PS, GW = K::GW, NXT = K::NXT, CW = K::CW;
    constexpr int AY1 = AY / 3;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ cplx smem[];
    cplx* twx = smem + NW * K::SLICE;             // W_NX^{n2 k1}, [k1][BPX]
    cplx* twx2 = K::TWX2 ? twx + K::TWX : twx;    // W_NX^{n1 k2} of the x-analysis split, [n1][BPX2]
    cplx* twy = twx + K::TWX + K::TWX2;           // W_NY^{k1 k2}, [k1][BY + 1]
    const uint32_t bars = smem_u32(twy + K::TWY);

    const int tid = threadIdx.x;
    const int lane0 = tid & 31;
    const int warp = __shfl_sync(FULL, tid >> 5, 0);
    cplx* A = smem + warp * K::SLICE;             // this warp's slice: x tile / pair storages
    const uint32_t ybar = bars + 8 * (uint32_t)warp;
    const int ngroup = gridDim.x / G, grp = blockIdx.x / G, rank = blockIdx.x % G;
    const int gw = rank * NW + warp;              // this warp within its group
    cplx* Zs = scratch + (size_t)grp * K::GROUP_SCRATCH_CPLX;   // [field][pair][row m + NX/2 | row m][cc]; field 0 = g
    cplx* Ps = Zs + NF * K::ZS_CPLX;                            // [pair][cc]
    unsigned* zcnt = cnt + 2 * grp;
    unsigned* pcnt = zcnt + 1;

    load_twiddles_ab<AX, BX>(twx, twx_g);
    if constexpr (K::TWX2 != 0) load_twiddles_ab<K::AX2, K::BX2>(twx2, twx_g);
    load_twiddles_ab<AY, BY>(twy, twy_g);
    if (tid == 0) {
        for (int w = 0; w < NW; ++w) mbar_init(bars + 8 * w, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();   // the only CTA-wide barrier of the kernel

    const unsigned T = (unsigned)nslab * (unsigned)nz * (unsigned)nv;   // planes of this launch (< 2^31: checked by the host)
    const size_t plane_elems = (size_t)NX0 * NKY0;
    // planes are walked v-fastest so that neighbouring groups share a chi plane in L2
    auto plane_of = [&](unsigned tt) {
        const unsigned v = tt % (unsigned)nv, zs = tt / (unsigned)nv;
        const unsigned z = zs % (unsigned)nz, sl = zs / (unsigned)nz;
        return (size_t)z + (size_t)nz * ((size_t)v + (size_t)nv * sl);
    };
    const uint64_t pol_keep = l2_policy_evict_last();
    // the columns of this warp's first X1 task of plane tt towards L2
    auto prefetch_x1 = [&](unsigned tt) {
        if (gw < NF * NXT) {
            const cplx* src = (CHIV && gw < NXT) ? chi : g;
            const int kyA = (gw % NXT) * CW, ncol = (kyA + CW + 1 <= NKY0) ? CW + 1 : CW;   // the -ky pair starts one column later
            wa_prefetch(src + plane_of(tt) * plane_elems + (size_t)kyA * NX0, sizeof(cplx) * ncol * NX0, lane0);
        }
    };
    if ((unsigned)grp < T) prefetch_x1((unsigned)grp);

    uint32_t yph = 0;
    unsigned it = 0;
    for (unsigned t = (unsigned)grp; t < T; t += (unsigned)ngroup, ++it) {
        const size_t p = plane_of(t);
        const size_t q = (size_t)((t / (unsigned)nv) % (unsigned)nz) + (size_t)nz * (size_t)(t / ((unsigned)nv * (unsigned)nz));
        cplx* Rb = rhs + p * plane_elems;
        [[maybe_unused]] const cplx* Rc = CHIV ? nullptr : R + q * ((size_t)NX * NY);
        [[maybe_unused]] const cplx* Rc2 = EM ? R2 + q * ((size_t)NX * NY) : nullptr;
        [[maybe_unused]] double vpar = 0.0;
        if constexpr (EM) vpar = __ldg(vp + (t % (unsigned)nv) + (unsigned)nv * (((unsigned)slab0 + t / ((unsigned)nv * (unsigned)nz)) / (unsigned)nw));

        // =============== X1: derivative, pad, x-synthesis; tasks (field, column pair) over the warps of the group ===============
#pragma unroll 1
        for (int task = gw; task < NF * NXT; task += GW) {
            const int lane = opaque(lane0);
            const bool is_chi = CHIV && task < NXT;   // with CHIV: chi first, then g
            const cplx* F = (is_chi ? chi : g) + p * plane_elems;
            cplx* Zf = Zs + (is_chi ? K::ZS_CPLX : 0);   // field 0 = g, field 1 = chi
            const int kyA = (task % NXT) * CW;
            if (task + GW < NF * NXT) {   // the next task's columns towards L2
                const int tn = task + GW, kyN = (tn % NXT) * CW, ncol = (kyN + CW + 1 <= NKY0) ? CW + 1 : CW;
                wa_prefetch(((CHIV && tn < NXT) ? chi : g) + p * plane_elems + (size_t)kyN * NX0, sizeof(cplx) * ncol * NX0, lane);
            }
            wa_x1_task<K, PF>(F, Zf, A, twx, kyA, lane, kxmin, kymin, pol_keep);
        }
        // ---- hand-over 1: every warp of the group has written its columns of Z ----
        wa_handover(zcnt, (unsigned)GW * (it + 1), lane0);

        // =============== Y: this CTA's row pairs, a warp takes NPW of them at a time, __syncwarp only ===============
        {
            const int lane = opaque(lane0);
            // the rhs columns of this warp's X2 tasks towards L2 (read after the second hand-over)
            for (int task = gw; task < NXT; task += GW) wa_prefetch(Rb + (size_t)(task * CW) * NX0, sizeof(cplx) * CW * NX0, lane);
            const int k1y = lane < AY ? lane : lane - AY;   // lanes >= AY shadow an item (same addresses) and skip the stores
            const bool act2 = lane < AY;
            const int j1 = (lane / BY) < NPW ? (lane / BY) : 0;   // Y1 / Y3 item: pair j1 of the warp item, position lane mod BY
            const bool act1 = (lane / BY) < NPW;
            const int n2 = lane % BY;
            constexpr bool TWREG = (BY == 8);                     // the lane's y twiddles in registers (else read at every use)
            cplx* Zw = A;                                         // this warp's pair storages: g, then (CHIV) chi
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
            // (dx chi, dy chi) of row `row` at y = k1 + AY k2, k2 < BY, from the real-space rows (EM: composed from two fields)
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
                    // after the hand-over) and this warp's tiles, which the copies overwrite (every item)
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
                // scratch exceeds what L2 keeps (768 x 384: 81 MB; DRAM writes 69 -> 34 GB per launch)
                if constexpr (K::GROUP_SCRATCH_CPLX * sizeof(cplx) > ((size_t)2 << 20)) {
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
                    for (int r = 0; r < NR; ++r) {  // Y2: twiddle + radix-BY to real space, bracket
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
                                cplx tw;
                                if constexpr (BY == 8) tw = FLAT ? tqr[k2] : tq[k2]; else tw = twl[k2];
                                w[k2] = cmul(w[k2], tw.x, -tw.y);
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
        // ---- hand-over 2: every warp of the group has written its rows of P ----
        wa_handover(pcnt, (unsigned)GW * (it + 1), lane0);

        // =============== X2: x-analysis; tasks (column pair) over the warps of the group ===============
        if (t + (unsigned)ngroup < T) prefetch_x1(t + (unsigned)ngroup);
#pragma unroll 1
        for (int task = gw; task < NXT; task += GW) {
            const int lane = opaque(lane0);
            wa_x2_task<K, PF>(Ps, Rb, A, twx2, task * CW, lane, coef, pol_keep);
        }
    }
}

}  // namespace gnl
