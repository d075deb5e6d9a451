// nl_fused.cuh -- one persistent kernel for the whole g-side of the hot path, a plane per CTA at a
// time, with the x<->y hand-over entirely in shared memory (no scratch traffic to L2/HBM).
//
// Used when the half-transformed plane Z (Nx x 2 nky0 complex) fits next to the exchange tiles in the
// 227 KB of one SM (configs[0], configs[1]); larger planes go through the batched kernels of
// nl_kernels.cuh.  Steps per plane:
//   X-inv : A1 derivative, A2 pad, x half of A3   g[ky][i]        -> Z[m][cc]   (in smem)
//   Y     : y half of A3, A4 bracket, y half of A5 Z rows, Rchi    -> P[pair][cc] (over Z, in place)
//   X-fwd : x half of A5, A6 delete/scale/add      P               -> rhs[ky][i] +=
// Rchi[q][m][y] = (dx chi, dy chi) comes from k_xinv + k_yreal (shared by the nv planes of a chi plane).
//
// Every length is N = A*8.  Warps work autonomously inside a phase (only __syncwarp); the three
// phases of a plane are separated by __syncthreads.  Exchange tiles of the two-stage FFTs live IN
// PLACE inside Z wherever the data they replace is already in registers:
//   * x columns: tile slot (k1,n2) of column cc sits in row 8 k1 + ((n2+k1)&7) of that column
//     (the skew keeps both the stage-1 stores and the stage-2 loads bank-conflict free);
//   * y rows: rows m and m+Nx/2 are stored side by side ("pair storage", 2*W2 slots + 1 pad); the
//     tile of the first row overwrites the pair storage, the tile of the second goes to a small
//     per-warp scratch tile.
#pragma once
#include <cuda_runtime.h>

#include "nl_kernels.cuh"

namespace gnl {

template <int AX, int AY, int NW>
struct Fused {
    static constexpr int NX = 8 * AX, NY = 8 * AY;
    static constexpr int NKY0 = NY / 3, W2 = 2 * NKY0, NPAIR = NX / 2, PS = 2 * W2 + 1;
    static constexpr int M = NX / 3, NX0 = 2 * M;
    static constexpr int FY = AY * 9;  // y tile [k1][9]
    static constexpr int ZSZ = NPAIR * PS;
    static constexpr int SMEM_CPLX = ZSZ + NW * 2 * FY + AX * 9 + AY * 9;
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)SMEM_CPLX;
    static constexpr int NJ = (4 * AX + 31) / 32;  // x items per lane when a warp does 4 columns
    static_assert(AX % 3 == 0 && AY % 3 == 0, "3/2 rule");
    static_assert(AY <= 16, "two pairs per Y2 pass need AY <= 16");

    // offset of row m of Z (rows m and m + NPAIR share one pair storage)
    __device__ static __forceinline__ int zrow(int m) { return (m % NPAIR) * PS + (m / NPAIR) * W2; }
    // offset of the 8-row group that holds the x tile slots (k1, *): rows 8 k1 .. 8 k1 + 7
    __device__ static __forceinline__ int tile_group(int k1)
    {
        if constexpr (NPAIR % 8 == 0) {
            const int half = (8 * k1 >= NPAIR) ? 1 : 0;
            return (8 * k1 - NPAIR * half) * PS + half * W2;
        } else {
            return -1;  // rows of a group may straddle the two halves: use zrow per row
        }
    }
    __device__ static __forceinline__ int tile_slot(int k1, int s)  // s = (n2 + k1) & 7
    {
        if constexpr (NPAIR % 8 == 0)
            return tile_group(k1) + s * PS;
        else
            return zrow(8 * k1 + s);
    }
};

// An opaque copy of a lane-constant value: keeps the compiler from hoisting per-lane address and
// wavenumber arithmetic out of the plane loop (where it would sit in registers for the whole kernel).
__device__ __forceinline__ int opaque(int v)
{
    asm volatile("" : "+r"(v));
    return v;
}

__device__ __forceinline__ void prefetch_l2(const void* p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// (i kx + kys) * f
__device__ __forceinline__ cplx deriv_mul(cplx f, double kx, double kys)
{
    return cmake(fma(kys, f.x, -kx * f.y), fma(kx, f.x, kys * f.y));
}

// X-inv stage 1 for one lane: column (kyi, sg), position n2.  KY0: the pass that contains ky = 0
// (Hermitian part of the ky = 0 column, reading R7; and the all-zero column cc = NKY0).
template <class C, int AX, bool KY0>
__device__ __forceinline__ void xinv_stage1(cplx* Z, const cplx* twx, const cplx* __restrict__ F, int u, int lane,
                                            double kxmin, double kymin)
{
    constexpr int AX1 = AX / 3, M = C::M, NX0 = C::NX0, W2 = C::W2, NKY0 = C::NKY0, PS = C::PS;
    const int n2 = lane & 7, sg = (lane >> 3) & 1, kyi = 2 * u + (lane >> 4);
    const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
    const cplx* Fc = F + (size_t)kyi * NX0 + n2;
    const double ky = kymin * (double)kyi;
    const double kys = sg ? ky : -ky;  // (i kx - ky) F for +ky, (i kx + ky) F for -ky
    const double dn2 = (double)n2;
    cplx lo[AX1], hi[AX1];
#pragma unroll
    for (int a = 0; a < AX1; ++a) {
        cplx f0 = Fc[8 * a], f1 = Fc[8 * a + M];
        if constexpr (KY0) {
            if (kyi == 0) {
                const int i0 = n2 + 8 * a, i1 = i0 + M;
                cplx m0 = F[(NX0 - i0) % NX0], m1 = F[NX0 - i1];
                f0 = cmake(0.5 * (f0.x + m0.x), 0.5 * (f0.y - m0.y));
                f1 = cmake(0.5 * (f1.x + m1.x), 0.5 * (f1.y - m1.y));
            }
        }
        const double kx0 = kxmin * (dn2 + (double)(8 * a));             // i = n2 + 8a        (kx >= 0)
        const double kx1 = kxmin * (dn2 + (double)(8 * a + M - NX0));   // i = n2 + 8a + M    (kx < 0)
        lo[a] = deriv_mul(f0, kx0, kys);
        hi[a] = deriv_mul(f1, kx1, kys);
        if (a == 0 && n2 == 0) hi[0] = cmake(0.0, 0.0);  // i = M: the Nyquist row is ignored (R6)
    }
    cplx out[AX];
    dft_pruned_in<AX, +1>(lo, hi, out);
    if constexpr (KY0) {
        if (sg && kyi == 0) {  // there is no -0 column: slot cc = NKY0 holds zeros
#pragma unroll
            for (int k1 = 0; k1 < AX; ++k1) out[k1] = cmake(0.0, 0.0);
        }
    }
    int soff[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) soff[r] = ((n2 + r) & 7) * PS + cc;
#pragma unroll
    for (int k1 = 0; k1 < AX; ++k1) {
        const cplx w = twx[k1 * 9 + n2];
        const cplx val = (k1 == 0) ? out[0] : cmul(out[k1], w.x, w.y);
        if constexpr (C::NPAIR % 8 == 0)
            Z[C::tile_group(k1) + soff[k1 & 7]] = val;
        else
            Z[C::zrow(8 * k1 + ((n2 + k1) & 7)) + cc] = val;
    }
}

template <int AX, int AY, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_plane_fused(const cplx* __restrict__ g, cplx* __restrict__ rhs, const cplx* __restrict__ R,
              const cplx* __restrict__ twx_g, const cplx* __restrict__ twy_g, int nz, int nv, int nslab,
              int chi_has_v, double kxmin, double kymin, double coef)
{
    using C = Fused<AX, AY, NW>;
    constexpr int NX = C::NX, NY = C::NY, NKY0 = C::NKY0, W2 = C::W2, NPAIR = C::NPAIR, PS = C::PS;
    constexpr int M = C::M, NX0 = C::NX0, FY = C::FY, NJ = C::NJ;
    constexpr int AX1 = AX / 3, AY1 = AY / 3;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ cplx smem[];
    cplx* Z = smem;
    cplx* ST = Z + C::ZSZ;
    cplx* twx = ST + NW * 2 * FY;
    cplx* twy = twx + AX * 9;
    const int lane0 = threadIdx.x & 31, warp = threadIdx.x >> 5;

    load_twiddles_ab<AX, 8>(twx, twx_g);
    load_twiddles_ab<AY, 8>(twy, twy_g);
    __syncthreads();

    const long long T = (long long)nslab * nz * nv;
    const size_t plane_elems = (size_t)NX0 * NKY0;
    for (long long t = blockIdx.x; t < T; t += gridDim.x) {
        // planes are walked v-fastest so that neighbouring CTAs share a chi plane in L2
        const int v = (int)(t % nv);
        const int z = (int)((t / nv) % nz);
        const long long sl = t / ((long long)nv * nz);
        const size_t p = (size_t)z + (size_t)nz * ((size_t)v + (size_t)nv * sl);
        const size_t q = chi_has_v ? p : (size_t)z + (size_t)nz * sl;
        const cplx* F = g + p * plane_elems;
        cplx* Rb = rhs + p * plane_elems;
        const cplx* Rc = R + q * ((size_t)NX * NY);
        {  // pull the next plane's g and rhs towards L2 while this one is being worked on
            const long long tn = t + gridDim.x;
            if (tn < T) {
                const int vn = (int)(tn % nv), zn = (int)((tn / nv) % nz);
                const long long sn = tn / ((long long)nv * nz);
                const size_t pn = (size_t)zn + (size_t)nz * ((size_t)vn + (size_t)nv * sn);
                const char* a = (const char*)(g + pn * plane_elems);
                const char* b = (const char*)(rhs + pn * plane_elems);
                for (size_t off = (size_t)threadIdx.x * 128; off < plane_elems * sizeof(cplx); off += (size_t)NW * 32 * 128) {
                    prefetch_l2(a + off);
                    prefetch_l2(b + off);
                }
            }
        }

        // ---------------- X-inv: 2 stored columns x {+ky, -ky} per warp pass --------------------
        for (int u = warp; u < NKY0 / 2; u += NW) {
            const int lane = opaque(lane0);
            if (u == 0)
                xinv_stage1<C, AX, true>(Z, twx, F, u, lane, kxmin, kymin);
            else
                xinv_stage1<C, AX, false>(Z, twx, F, u, lane, kxmin, kymin);
            __syncwarp(FULL);
            // stage 2: every lane first reads ALL its tile slots (the outputs overwrite the same column)
            cplx vv[NJ][8];
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int item = lane + 32 * j;
                if (item < 4 * AX) {
                    const int cidx = item / AX, k1 = item % AX;
                    const int sg = cidx & 1, kyi = 2 * u + (cidx >> 1);
                    const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
                    if constexpr (NPAIR % 8 == 0) {
                        const cplx* Zt = Z + C::tile_group(k1) + cc;
#pragma unroll
                        for (int n2 = 0; n2 < 8; ++n2) vv[j][n2] = Zt[((n2 + k1) & 7) * PS];
                    } else {
#pragma unroll
                        for (int n2 = 0; n2 < 8; ++n2) vv[j][n2] = Z[C::zrow(8 * k1 + ((n2 + k1) & 7)) + cc];
                    }
                }
            }
            __syncwarp(FULL);
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int item = lane + 32 * j;
                if (item < 4 * AX) {
                    const int cidx = item / AX, k1 = item % AX;
                    const int sg = cidx & 1, kyi = 2 * u + (cidx >> 1);
                    const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
                    Dft<8, +1>::run(vv[j]);
                    cplx* Zo = Z + k1 * PS + cc;  // row k1 + AX*k2: first half for k2 < 4 (k1 < AX, NPAIR = 4 AX)
                    const double sgn = sg ? -1.0 : 1.0;
#pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2)
                        Zo[(k2 < 4) ? AX * k2 * PS : AX * (k2 - 4) * PS + W2] = cmake(vv[j][k2].x, sgn * vv[j][k2].y);
                }
            }
        }
        __syncthreads();

        // ---------------- Y: two row pairs (m, m + NX/2) per warp pass ---------------------------
        for (int u = warp; u < NPAIR / 2; u += NW) {
            const int lane = opaque(lane0);
            // chi values of this lane's Y2 item, requested now so that their latency hides behind Y1
            const int pidx2 = lane >> 4, k1y = lane & 15;
            const bool act2 = k1y < AY;
            const int pair2 = 2 * u + pidx2;
            cplx chv[2][8];
            if (act2) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const cplx* Rr = Rc + (size_t)(pair2 + h * NPAIR) * NY + k1y;
#pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2) chv[h][k2] = __ldg(Rr + AY * k2);
                }
            }
            {  // Y1: pruned radix-AY + twiddle, 4 rows x 8 lanes
                const int ridx = lane >> 3, n2 = lane & 7;
                const int pair1 = 2 * u + (ridx >> 1), h1 = ridx & 1;
                const cplx* Zr = Z + pair1 * PS + h1 * W2 + n2;
                cplx lo[AY1], hi[AY1], tw[AY];
#pragma unroll
                for (int a = 0; a < AY1; ++a) {
                    lo[a] = Zr[8 * a];
                    hi[a] = Zr[8 * a + NKY0];
                }
#pragma unroll
                for (int k1 = 1; k1 < AY; ++k1) tw[k1] = twy[k1 * 9 + n2];
                cplx out[AY];
                dft_pruned_in<AY, +1>(lo, hi, out);
                __syncwarp(FULL);  // every lane has read its row before the tiles overwrite the pair storage
                cplx* tile = (h1 ? ST + (warp * 2 + (ridx >> 1)) * FY : Z + pair1 * PS) + n2;
                tile[0] = out[0];
#pragma unroll
                for (int k1 = 1; k1 < AY; ++k1) tile[k1 * 9] = cmul(out[k1], tw[k1].x, tw[k1].y);
            }
            __syncwarp(FULL);
            if (act2) {  // Y2: to real space (both rows), bracket, back; result replaces tile 0 in place
                cplx* tile0 = Z + pair2 * PS + k1y * 9;
                const cplx* tile1 = ST + (warp * 2 + pidx2) * FY + k1y * 9;
                cplx v0[8], v1[8], tq[8];
#pragma unroll
                for (int n2 = 0; n2 < 8; ++n2) v0[n2] = tile0[n2];
#pragma unroll
                for (int n2 = 0; n2 < 8; ++n2) v1[n2] = tile1[n2];
#pragma unroll
                for (int k2 = 1; k2 < 8; ++k2) tq[k2] = twy[k1y * 9 + k2];
                Dft<8, +1>::run(v0);
                Dft<8, +1>::run(v1);
                cplx w[8];
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) {  // dx chi * dy g - dy chi * dx g for rows m and m + NX/2
                    w[k2].x = fma(chv[0][k2].x, v0[k2].y, -chv[0][k2].y * v0[k2].x);
                    w[k2].y = fma(chv[1][k2].x, v1[k2].y, -chv[1][k2].y * v1[k2].x);
                }
                Dft<8, -1>::run(w);
                tile0[0] = w[0];
#pragma unroll
                for (int k2 = 1; k2 < 8; ++k2) tile0[k2] = cmul(w[k2], tq[k2].x, -tq[k2].y);
            }
            __syncwarp(FULL);
            {  // Y3: pruned-output radix-AY; P[pair][cc] overwrites tile 0 after everyone has read it
                const bool act3 = lane < 16;
                const int pair3 = 2 * u + ((lane >> 3) & 1), k2 = lane & 7;
                cplx in[AY];
                if (act3) {
#pragma unroll
                    for (int n1 = 0; n1 < AY; ++n1) in[n1] = Z[pair3 * PS + n1 * 9 + k2];
                }
                __syncwarp(FULL);
                if (act3) {
                    cplx lo[AY1], hi[AY1];
                    dft_pruned_out<AY, -1>(in, lo, hi);
                    cplx* Pp = Z + pair3 * PS + k2;
#pragma unroll
                    for (int c = 0; c < AY1; ++c) {
                        Pp[8 * c] = lo[c];
                        Pp[8 * c + NKY0] = hi[c];
                    }
                }
            }
        }
        __syncthreads();

        // ---------------- X-fwd: 4 stored columns per warp pass ----------------------------------
        for (int u = warp; u < NKY0 / 4; u += NW) {
            const int lane = opaque(lane0);
            cplx xx[NJ][8];
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int item = lane + 32 * j;
                if (item < 4 * AX) {
                    const int col = item / AX, n1 = item % AX;
                    const int kyi = 4 * u + col;
                    const cplx* Pp = Z + n1 * PS + kyi;
                    const cplx* Pm = Z + n1 * PS + (kyi ? W2 - kyi : 0);
#pragma unroll
                    for (int n2 = 0; n2 < 4; ++n2) {  // rows m = n1 + AX n2 and m + NX/2 of pair n1 + AX n2
                        const cplx pp = Pp[AX * n2 * PS], pm = Pm[AX * n2 * PS];
                        xx[j][n2] = cmake(pp.x + pm.x, pp.y - pm.y);      // 2 N^_m  = P+ + conj P-
                        xx[j][n2 + 4] = cmake(pp.y + pm.y, pm.x - pp.x);  // 2 N^_m' = -i (P+ - conj P-)
                    }
                }
            }
            __syncwarp(FULL);
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int item = lane + 32 * j;
                if (item < 4 * AX) {
                    const int col = item / AX, n1 = item % AX;
                    const int kyi = 4 * u + col;
                    const int s0 = kyi, s1 = kyi ? W2 - kyi : NKY0;
                    cplx tq[8];
#pragma unroll
                    for (int k2 = 1; k2 < 8; ++k2) tq[k2] = twx[n1 * 9 + k2];
                    Dft<8, -1>::run(xx[j]);
                    if constexpr (NPAIR % 8 == 0) {
                        // tile slot (n1,k2) -> row 8 n1 + ((k2+n1)&7); second-half rows use slot s1 of their pair
                        const int half = (8 * n1 >= NPAIR) ? 1 : 0;
                        cplx* Zt = Z + (8 * n1 - NPAIR * half) * PS + (half ? s1 : s0);
                        Zt[(n1 & 7) * PS] = xx[j][0];
#pragma unroll
                        for (int k2 = 1; k2 < 8; ++k2)
                            Zt[((k2 + n1) & 7) * PS] = cmul(xx[j][k2], tq[k2].x, -tq[k2].y);
                    } else {
#pragma unroll
                        for (int k2 = 0; k2 < 8; ++k2) {
                            const int e = 8 * n1 + ((k2 + n1) & 7);
                            Z[(e % NPAIR) * PS + ((e / NPAIR) ? s1 : s0)] =
                                (k2 == 0) ? xx[j][0] : cmul(xx[j][k2], tq[k2].x, -tq[k2].y);
                        }
                    }
                }
            }
            __syncwarp(FULL);
            {
                const int col = lane >> 3, k2 = lane & 7;
                const int kyi = 4 * u + col;
                const int s0 = kyi, s1 = kyi ? W2 - kyi : NKY0;
                cplx in[AX];
                if constexpr (NPAIR % 8 == 0) {
                    int soff[8];
#pragma unroll
                    for (int r = 0; r < 8; ++r) soff[r] = ((k2 + r) & 7) * PS;
#pragma unroll
                    for (int n1 = 0; n1 < AX; ++n1) {
                        const int half = (8 * n1 >= NPAIR) ? 1 : 0;
                        in[n1] = Z[(8 * n1 - NPAIR * half) * PS + soff[n1 & 7] + (half ? s1 : s0)];
                    }
                } else {
#pragma unroll
                    for (int n1 = 0; n1 < AX; ++n1) {
                        const int e = 8 * n1 + ((k2 + n1) & 7);
                        in[n1] = Z[(e % NPAIR) * PS + ((e / NPAIR) ? s1 : s0)];
                    }
                }
                cplx lo[AX1], hi[AX1];
                dft_pruned_out<AX, -1>(in, lo, hi);
                cplx* Rcol = Rb + (size_t)kyi * NX0 + k2;
#pragma unroll
                for (int c = 0; c < AX1; ++c) {  // delete the padded modes, prefactor, add to rhs
                    const cplx r0 = Rcol[8 * c];
                    Rcol[8 * c] = cmake(fma(coef, lo[c].x, r0.x), fma(coef, lo[c].y, r0.y));
                    if (c != 0 || k2 != 0) {  // i = M is the Nyquist row: untouched (R6)
                        const cplx r1 = Rcol[8 * c + M];
                        Rcol[8 * c + M] = cmake(fma(coef, hi[c].x, r1.x), fma(coef, hi[c].y, r1.y));
                    }
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace gnl
