// nl_fused2.cuh -- second-generation fused per-plane kernel (planes whose half-transformed form Z fits
// one SM's shared memory and whose ky extent fills whole warps: nky0 a multiple of 32).
//
// Same steps as nl_fused.cuh, re-laid-out around what the ncu
// capture of the first kernel showed: its L1/shared-memory data pipe (1 wavefront of 128 B per clock)
// was busier than the FP64 pipe, a quarter of that traffic being per-lane twiddle loads.  Here
//   * the x exchange tile lives IN PLACE in the rows a stage-2 thread both reads and writes
//     (slot (k1,n2) of column cc sits in row k1 + AX n2, at column cc ^ n2 -- the xor keeps the
//     stage-1 stores, whose lanes run over n2, bank-conflict free), so stage 2 needs no read-all-
//     then-write ordering and no per-warp ownership of columns;
//   * the lanes of x stage 2 (both directions) run over 32 columns with k1 (n1) uniform in the warp,
//     so its twiddles W_Nx^{n2 k1} are warp-uniform: they come from constant memory through the
//     uniform datapath and cost neither registers nor shared-memory wavefronts;
//   * the y twiddles W_Ny^{k1 k2} are applied on the k1 side (Y2), where they depend on the lane only:
//     7 complex values per lane per plane serve the two inverse rows and (conjugated) the forward row;
//   * g is read once per column (the +ky and -ky syntheses share the loads), rhs values are requested
//     before the last x stage so their latency hides behind it, Y3 runs on 4 pairs with all 32 lanes.
//   * for one k1, x stage 2, the y work of 4 row pairs and the first x stage of the way back touch the same 4 pair
//     storages and nothing else: a warp runs such a chain with __syncwarp only, so a plane needs 3 __syncthreads
//     (after the first and before/after the last pruned radix-AX stage) and warps drift apart inside the chains,
//     which lets the FP64 pipe of one overlap the shared-memory traffic of another.
#pragma once
#include <cuda_runtime.h>

#include "nl_fused.cuh"

namespace gnl {

// W_N^j for every supported transform length N, back to back (filled by gene_nl_create)
constexpr int kCTwTotal = 24 + 48 + 96 + 144 + 192 + 384 + 768;
__constant__ cplx c_tw[kCTwTotal];
__host__ __device__ constexpr int ctw_offset(int n)
{
    return n == 24 ? 0 : n == 48 ? 24 : n == 96 ? 72 : n == 144 ? 168 : n == 192 ? 312 : n == 384 ? 504 : n == 768 ? 888 : -1;
}

// 128-bit global loads the compiler may not sink below later shared-memory work (they are issued where
// they are written, ahead of the butterflies that hide their latency)
__device__ __forceinline__ cplx ldg_nc_early(const cplx* p)
{
    cplx v;
    asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ cplx ldg_early(const cplx* p)
{
    cplx v;
    asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}

template <int AX, int AY, int NW>
struct Fused2 {
    static constexpr int NX = 8 * AX, NY = 8 * AY;
    static constexpr int NKY0 = NY / 3, W2 = 2 * NKY0, NPAIR = NX / 2, PS = 2 * W2 + 1;
    static constexpr int M = NX / 3, NX0 = 2 * M;
    static constexpr int FY = AY * 9;  // y tile [k1][9]
    static constexpr int ZSZ = NPAIR * PS;
    static constexpr int SMEM_CPLX = ZSZ + NW * 2 * FY + AY * 9;
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)SMEM_CPLX;
    static constexpr int OFFX = ctw_offset(NX);
    static_assert(AX % 3 == 0 && AY % 3 == 0, "3/2 rule");
    static_assert(NKY0 % 32 == 0, "lanes of the x stage 2 run over 32 stored columns");
    static_assert(AY <= 16, "two pairs per Y2 pass need AY <= 16");
    static_assert(NPAIR == 4 * AX && OFFX >= 0, "geometry");
    // offset of x-tile row k1 + AX*n2 (relative to row k1): rows n2 < 4 are first halves of pair storages
    __device__ static __forceinline__ int xrow(int n2) { return (AX * (n2 & 3)) * PS + (n2 >> 2) * W2; }
};

template <int AX, int AY, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_plane_fused2(const cplx* __restrict__ g, cplx* __restrict__ rhs, const cplx* __restrict__ R,
               const cplx* __restrict__ twy_g, int nz, int nv, int nslab, int chi_has_v, double kxmin, double kymin,
               double coef)
{
    using C = Fused2<AX, AY, NW>;
    constexpr int NX = C::NX, NY = C::NY, NKY0 = C::NKY0, W2 = C::W2, NPAIR = C::NPAIR, PS = C::PS;
    constexpr int M = C::M, NX0 = C::NX0, FY = C::FY, OFFX = C::OFFX;
    constexpr int AX1 = AX / 3, AY1 = AY / 3;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ cplx smem[];
    cplx* Z = smem;
    cplx* ST = Z + C::ZSZ;
    cplx* twy = ST + NW * 2 * FY;
    const int lane0 = threadIdx.x & 31;
    const int warp = __shfl_sync(FULL, (int)(threadIdx.x >> 5), 0);  // provably warp-uniform

    load_twiddles_ab<AY, 8>(twy, twy_g);
    __syncthreads();

    static_assert(NKY0 / 4 == NW, "one pruned radix-AX pass (4 stored columns) per warp");
    const long long T = (long long)nslab * nz * nv;
    const size_t plane_elems = (size_t)NX0 * NKY0;
    // planes are walked v-fastest so that neighbouring CTAs share a chi plane in L2
    auto plane_of = [&](long long tt) {
        const int v = (int)(tt % nv);
        const int z = (int)((tt / nv) % nz);
        const long long sl = tt / ((long long)nv * nz);
        return (size_t)z + (size_t)nz * ((size_t)v + (size_t)nv * sl);
    };
    // This warp's share of a spectral plane for the first x stage (column kyi = 4 warp + lane/8, rows n2 + 8a and
    // n2 + 8a + M).  Requested one barrier ahead of its use: for the first plane here, for later planes at the end of
    // the previous one, so that the L2 latency hides behind the warps that are still working.
    cplx f0[AX1], f1[AX1];
    auto request_g = [&](long long tt) {
        const int lane = opaque(lane0);
        const int n2 = lane & 7, kyi = 4 * warp + (lane >> 3);
        const cplx* F = g + plane_of(tt) * plane_elems;
        const cplx* Fc = F + (size_t)kyi * NX0 + n2;
#pragma unroll
        for (int a = 0; a < AX1; ++a) {
            f0[a] = ldg_nc_early(Fc + 8 * a);
            f1[a] = ldg_nc_early(Fc + 8 * a + M);
        }
        if (kyi == 0) {  // Hermitian part of the ky = 0 column (reading R7)
#pragma unroll
            for (int a = 0; a < AX1; ++a) {
                const int i0 = n2 + 8 * a, i1 = i0 + M;
                const cplx m0 = F[(NX0 - i0) % NX0], m1 = F[NX0 - i1];
                f0[a] = cmake(0.5 * (f0[a].x + m0.x), 0.5 * (f0[a].y - m0.y));
                f1[a] = cmake(0.5 * (f1[a].x + m1.x), 0.5 * (f1[a].y - m1.y));
            }
        }
        if (n2 == 0) f1[0] = cmake(0.0, 0.0);  // i = M: the Nyquist row is ignored (R6)
    };
    if ((long long)blockIdx.x < T) request_g(blockIdx.x);
    for (long long t = blockIdx.x; t < T; t += gridDim.x) {
        const size_t p = plane_of(t);
        const size_t q = chi_has_v ? p : (size_t)((t / nv) % nz) + (size_t)nz * (size_t)(t / ((long long)nv * nz));
        cplx* Rb = rhs + p * plane_elems;
        const cplx* Rc = R + q * ((size_t)NX * NY);
        {  // pull the next plane's g and rhs towards L2 while this one is being worked on
            const long long tn = t + gridDim.x;
            if (tn < T) {
                const size_t pn = plane_of(tn);
                if (threadIdx.x == 0) {   // one bulk prefetch per array (TMA, SASS UBLKPF) instead of a line-by-line loop (-0.5 %)
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(g + pn * plane_elems), "r"((uint32_t)(plane_elems * sizeof(cplx))) : "memory");
                    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(rhs + pn * plane_elems), "r"((uint32_t)(plane_elems * sizeof(cplx))) : "memory");
                }
            }
        }

        // ------ X-inv stage 1: derivative, pad, pruned radix-AX; 4 stored columns x 8 n2 per warp ------
        {
            const int lane = opaque(lane0);
            const int n2 = lane & 7, kyi = 4 * warp + (lane >> 3);
            const double ky = kymin * (double)kyi, dn2 = (double)n2;
            cplx* Zl = Z + C::xrow(n2);
#pragma unroll 1
            for (int sg = 0; sg < 2; ++sg) {
                const double kys = sg ? ky : -ky;  // (i kx - ky) F for +ky, (i kx + ky) F for -ky
                const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
                cplx lo[AX1], hi[AX1];
#pragma unroll
                for (int a = 0; a < AX1; ++a) {
                    const double kx0 = kxmin * (dn2 + (double)(8 * a));            // i = n2 + 8a      (kx >= 0)
                    const double kx1 = kxmin * (dn2 + (double)(8 * a + M - NX0));  // i = n2 + 8a + M  (kx < 0)
                    lo[a] = deriv_mul(f0[a], kx0, kys);
                    hi[a] = deriv_mul(f1[a], kx1, kys);
                }
                cplx out[AX];
                dft_pruned_in<AX, +1>(lo, hi, out);
                if (sg && kyi == 0) {  // there is no -0 column: slot cc = NKY0 holds zeros
#pragma unroll
                    for (int k1 = 0; k1 < AX; ++k1) out[k1] = cmake(0.0, 0.0);
                }
                cplx* Zc = Zl + (cc ^ n2);
#pragma unroll
                for (int k1 = 0; k1 < AX; ++k1) Zc[k1 * PS] = out[k1];
            }
        }
        __syncthreads();

        // ------ chains: everything between the two pruned radix-AX stages touches, for one k1 (= n1), only the
        // pair storages k1 + AX j (j < 4): x stage 2 (rows k1 + AX n2), the y transforms and the bracket of those
        // 4 pairs, and the first x stage of the way back.  A warp runs whole chains; only __syncwarp inside ------
        {
            const int lane = opaque(lane0);
            // Y2 item of this lane: pair pidx2 of the pass, k1 = k1y.  Lanes with (lane & 15) >= AY shadow an item
            // of their own quarter-warp (same addresses: broadcast) and only skip the final stores, so the phase
            // has no divergent region
            const int pidx2 = lane >> 4;
            const bool act2 = (lane & 15) < AY;
            const int k1y = act2 ? (lane & 15) : 8 + (lane & 3);
            cplx tq[8];  // W_NY^{k1y k2}: twiddles of this lane's Y2 items (inverse rows; conjugated on the way back)
#pragma unroll
            for (int k2 = 1; k2 < 8; ++k2) tq[k2] = twy[k1y * 9 + k2];

            for (int c = warp; c < AX; c += NW) {
                cplx* Zc = Z + c * PS;  // pair storage c; pair c + AX j is j*AX*PS further
                // chi values of the first Y2 pass, requested now: their latency hides behind x stage 2 and Y1
                cplx chv[2][8];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const cplx* Rr = Rc + (size_t)(c + AX * pidx2 + h * NPAIR) * NY + k1y;
#pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2) chv[h][k2] = ldg_nc_early(Rr + AY * k2);
                }
                // -- x stage 2: twiddle (warp-uniform) + radix-8, in place; lanes over 32 columns --
                {
                    cplx vv[W2 / 32][8];
#pragma unroll
                    for (int grp = 0; grp < W2 / 32; ++grp) {
                        const int cc = 32 * grp + lane;
#pragma unroll
                        for (int n2 = 0; n2 < 8; ++n2) vv[grp][n2] = Zc[C::xrow(n2) + (cc ^ n2)];
                    }
#pragma unroll
                    for (int grp = 0; grp < W2 / 32; ++grp) {
                        const int cc = 32 * grp + lane;
                        cplx wx[8];
                        wx[0] = cmake(1.0, 0.0);
#pragma unroll
                        for (int n2 = 1; n2 < 8; ++n2) wx[n2] = c_tw[OFFX + n2 * c];
                        dft8_twiddled<+1>(vv[grp], wx);
                        const double sgn = (32 * grp >= NKY0) ? -1.0 : 1.0;  // -ky columns hold the conjugate
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2)
                            Zc[C::xrow(k2) + (cc ^ k2)] = cmake(vv[grp][k2].x, sgn * vv[grp][k2].y);
                    }
                }
                __syncwarp(FULL);
                // now Z[m][cc], m = c + AX k2, sits in pair storage c + AX (k2 & 3), half k2 >> 2, column cc ^ k2

                // -- y: pass 0 on pairs c, c + AX; pass 1 on pairs c + 2 AX, c + 3 AX --
#pragma unroll 1
                for (int pass = 0; pass < 2; ++pass) {
                    if (pass) {
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const cplx* Rr = Rc + (size_t)(c + AX * (2 + pidx2) + h * NPAIR) * NY + k1y;
#pragma unroll
                            for (int k2 = 0; k2 < 8; ++k2) chv[h][k2] = ldg_nc_early(Rr + AY * k2);
                        }
                    }
                    {  // Y1: pruned radix-AY, 4 rows x 8 lanes
                        const int ridx = lane >> 3, n2 = lane & 7;
                        const int j1 = 2 * pass + (ridx >> 1), h1 = ridx & 1;
                        const int sw = j1 + 4 * h1;  // column swizzle of row c + AX (j1 + 4 h1)
                        const cplx* Zr = Zc + j1 * (AX * PS) + h1 * W2 + (n2 ^ sw);
                        cplx lo[AY1], hi[AY1];
#pragma unroll
                        for (int a = 0; a < AY1; ++a) {
                            lo[a] = Zr[8 * a];
                            hi[a] = Zr[8 * a + NKY0];
                        }
                        cplx out[AY];
                        dft_pruned_in<AY, +1>(lo, hi, out);
                        __syncwarp(FULL);  // every lane has read its row before the tiles overwrite the pair storage
                        cplx* tile = (h1 ? ST + (warp * 2 + (ridx >> 1)) * FY : Zc + j1 * (AX * PS)) + n2;
#pragma unroll
                        for (int k1 = 0; k1 < AY; ++k1) tile[k1 * 9] = out[k1];
                    }
                    __syncwarp(FULL);
                    {  // Y2: twiddle, to real space (both rows), bracket, back; result replaces tile 0 in place
                        cplx* tile0 = Zc + (2 * pass + pidx2) * (AX * PS) + k1y * 9;
                        const cplx* tile1 = ST + (warp * 2 + pidx2) * FY + k1y * 9;
                        cplx v0[8], v1[8];
#pragma unroll
                        for (int n2 = 0; n2 < 8; ++n2) v0[n2] = tile0[n2];
#pragma unroll
                        for (int n2 = 0; n2 < 8; ++n2) v1[n2] = tile1[n2];
                        dft8_twiddled<+1>(v0, tq);
                        dft8_twiddled<+1>(v1, tq);
                        cplx w[8];
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2) {  // dx chi * dy g - dy chi * dx g for rows m and m + NX/2
                            w[k2].x = fma(chv[0][k2].x, v0[k2].y, -chv[0][k2].y * v0[k2].x);
                            w[k2].y = fma(chv[1][k2].x, v1[k2].y, -chv[1][k2].y * v1[k2].x);
                        }
                        Dft<8, -1>::run(w);
#pragma unroll
                        for (int k2 = 1; k2 < 8; ++k2) w[k2] = cmul(w[k2], tq[k2].x, -tq[k2].y);
                        __syncwarp(FULL);  // shadow lanes have read their tiles before the owners overwrite them
                        if (act2) {
#pragma unroll
                            for (int k2 = 0; k2 < 8; ++k2) tile0[k2] = w[k2];
                        }
                    }
                    __syncwarp(FULL);
                }
                {  // Y3: pruned-output radix-AY on the 4 pairs; P[pair][cc] overwrites tile 0 after everyone has read it
                    const int k2 = lane & 7;
                    cplx* Pp = Zc + (lane >> 3) * (AX * PS) + k2;
                    cplx in[AY];
#pragma unroll
                    for (int n1 = 0; n1 < AY; ++n1) in[n1] = Pp[n1 * 9];
                    __syncwarp(FULL);
                    cplx lo[AY1], hi[AY1];
                    dft_pruned_out<AY, -1>(in, lo, hi);
#pragma unroll
                    for (int cq = 0; cq < AY1; ++cq) {
                        Pp[8 * cq] = lo[cq];
                        Pp[8 * cq + NKY0] = hi[cq];
                    }
                }
                __syncwarp(FULL);

                // -- x stage 1 of the way back: unpack the row pair, radix-8, twiddle (warp-uniform); lanes over 32
                // columns.  Tile slot (kyi, n1 = c, k2) goes to the free second half of pair storage c + AX (k2 & 3) --
#pragma unroll
                for (int kg = 0; kg < NKY0 / 32; ++kg) {
                    const int kyi = 32 * kg + lane;
                    const cplx* Pq = Zc + kyi;
                    const cplx* Pm = Zc + (kyi ? W2 - kyi : 0);
                    cplx xx[8];
#pragma unroll
                    for (int n2 = 0; n2 < 4; ++n2) {  // rows m = c + AX n2 and m + NX/2 of pair c + AX n2
                        const cplx pp = Pq[AX * n2 * PS], pm = Pm[AX * n2 * PS];
                        xx[n2] = cmake(pp.x + pm.x, pp.y - pm.y);      // 2 N^_m  = P+ + conj P-
                        xx[n2 + 4] = cmake(pp.y + pm.y, pm.x - pp.x);  // 2 N^_m' = -i (P+ - conj P-)
                    }
                    Dft<8, -1>::run(xx);
                    cplx* Zt = Zc + W2;
                    Zt[kyi] = xx[0];
#pragma unroll
                    for (int k2 = 1; k2 < 8; ++k2) {
                        const cplx w = c_tw[OFFX + c * k2];
                        Zt[(AX * (k2 & 3)) * PS + NKY0 * (k2 >> 2) + (kyi ^ k2)] = cmul(xx[k2], w.x, -w.y);
                    }
                }
            }
        }
        // rhs values of this warp's share of the last stage, requested ahead of the barrier: the warps that finish
        // their chains first hide the latency behind the others
        cplx r0[AX1], r1[AX1];
        {
            const int lane = opaque(lane0);
            const cplx* Rcol = Rb + (size_t)(4 * warp + (lane >> 3)) * NX0 + (lane & 7);
#pragma unroll
            for (int c = 0; c < AX1; ++c) {
                r0[c] = ldg_early(Rcol + 8 * c);
                r1[c] = ldg_early(Rcol + 8 * c + M);
            }
        }
        __syncthreads();
        // next plane's share of g, requested here: the last x stage and the rhs update hide its latency
        if (t + gridDim.x < T) request_g(t + gridDim.x);

        // ------ X-fwd stage 2: pruned-output radix-AX, delete modes, prefactor, add; 4 columns x 8 k2 per warp ------
        {
            const int lane = opaque(lane0);
            const int k2 = lane & 7, kyi = 4 * warp + (lane >> 3);
            cplx* Rcol = Rb + (size_t)kyi * NX0 + k2;
            const cplx* Zt = Z + W2 + (AX * (k2 & 3)) * PS + NKY0 * (k2 >> 2) + (kyi ^ k2);
            cplx in[AX];
#pragma unroll
            for (int n1 = 0; n1 < AX; ++n1) in[n1] = Zt[n1 * PS];
            cplx lo[AX1], hi[AX1];
            dft_pruned_out<AX, -1>(in, lo, hi);
#pragma unroll
            for (int c = 0; c < AX1; ++c) {  // delete the padded modes, prefactor, add to rhs
                Rcol[8 * c] = cmake(fma(coef, lo[c].x, r0[c].x), fma(coef, lo[c].y, r0[c].y));
                if (c != 0 || k2 != 0)  // i = M is the Nyquist row: untouched (R6)
                    Rcol[8 * c + M] = cmake(fma(coef, hi[c].x, r1[c].x), fma(coef, hi[c].y, r1[c].y));
            }
        }
        __syncthreads();
    }
}

}  // namespace gnl
