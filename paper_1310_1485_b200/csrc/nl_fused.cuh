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

    __device__ static __forceinline__ int zrow(int m) { return (m % NPAIR) * PS + (m / NPAIR) * W2; }
};

__device__ __forceinline__ cplx ldg_nc(const cplx* p)
{
    return __ldg(p);
}

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
            {
                const int n2 = lane & 7, sg = (lane >> 3) & 1, kyi = 2 * u + (lane >> 4);
                const bool zero = sg && kyi == 0;  // there is no -0 column: slot cc = NKY0 holds zeros
                const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
                const cplx* Fc = F + (size_t)kyi * NX0;
                const double ky = kymin * (double)kyi;
                const double kys = sg ? ky : -ky;
                cplx lo[AX1], hi[AX1];
#pragma unroll
                for (int a = 0; a < AX1; ++a) {
                    {
                        const int i = n2 + 8 * a;
                        const double kx = kxmin * (double)i;
                        cplx f = Fc[i];
                        if (kyi == 0) {
                            cplx fm = Fc[(NX0 - i) % NX0];
                            f = cmake(0.5 * (f.x + fm.x), 0.5 * (f.y - fm.y));
                        }
                        lo[a] = cmake(fma(kys, f.x, -kx * f.y), fma(kx, f.x, kys * f.y));
                    }
                    {
                        const int i = n2 + 8 * a + M;
                        const double kx = kxmin * (double)(i - NX0);
                        cplx f = Fc[i];
                        if (kyi == 0) {
                            cplx fm = Fc[NX0 - i];
                            f = cmake(0.5 * (f.x + fm.x), 0.5 * (f.y - fm.y));
                        }
                        cplx val = cmake(fma(kys, f.x, -kx * f.y), fma(kx, f.x, kys * f.y));
                        hi[a] = (i == M) ? cmake(0.0, 0.0) : val;
                    }
                }
                cplx out[AX];
                dft_pruned_in<AX, +1>(lo, hi, out);
#pragma unroll
                for (int k1 = 0; k1 < AX; ++k1) {
                    const int row = 8 * k1 + ((n2 + k1) & 7);
                    cplx w = twx[k1 * 9 + n2];
                    cplx val = (k1 == 0) ? out[0] : cmul(out[k1], w.x, w.y);
                    Z[C::zrow(row) + cc] = zero ? cmake(0.0, 0.0) : val;
                }
            }
            __syncwarp(FULL);
            cplx vv[NJ][8];
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int item = lane + 32 * j;
                if (item < 4 * AX) {
                    const int cidx = item / AX, k1 = item % AX;
                    const int sg = cidx & 1, kyi = 2 * u + (cidx >> 1);
                    const int cc = sg ? (kyi ? W2 - kyi : NKY0) : kyi;
#pragma unroll
                    for (int n2 = 0; n2 < 8; ++n2) vv[j][n2] = Z[C::zrow(8 * k1 + ((n2 + k1) & 7)) + cc];
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
#pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2)
                        Z[C::zrow(k1 + AX * k2) + cc] = sg ? cconj(vv[j][k2]) : vv[j][k2];
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
                    for (int k2 = 0; k2 < 8; ++k2) chv[h][k2] = ldg_nc(Rr + AY * k2);
                }
            }
            {  // Y1: pruned radix-AY + twiddle, 4 rows x 8 lanes
                const int ridx = lane >> 3, n2 = lane & 7;
                const int pair1 = 2 * u + (ridx >> 1), h1 = ridx & 1;
                const cplx* Zr = Z + pair1 * PS + h1 * W2;
                cplx lo[AY1], hi[AY1];
#pragma unroll
                for (int a = 0; a < AY1; ++a) {
                    lo[a] = Zr[n2 + 8 * a];
                    hi[a] = Zr[n2 + 8 * a + NKY0];
                }
                cplx out[AY];
                dft_pruned_in<AY, +1>(lo, hi, out);
                __syncwarp(FULL);  // every lane has read its row before the tiles overwrite the pair storage
                cplx* tile = h1 ? ST + (warp * 2 + (ridx >> 1)) * FY : Z + pair1 * PS;
#pragma unroll
                for (int k1 = 0; k1 < AY; ++k1) {
                    cplx w = twy[k1 * 9 + n2];
                    tile[k1 * 9 + n2] = (k1 == 0) ? out[0] : cmul(out[k1], w.x, w.y);
                }
            }
            __syncwarp(FULL);
            if (act2) {  // Y2: to real space (both rows), bracket, back; result replaces tile 0 in place
                cplx w[8];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const cplx* tile = h ? ST + (warp * 2 + pidx2) * FY : Z + pair2 * PS;
                    cplx vr[8];
#pragma unroll
                    for (int n2 = 0; n2 < 8; ++n2) vr[n2] = tile[k1y * 9 + n2];
                    Dft<8, +1>::run(vr);
#pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2) {
                        const cplx c = chv[h][k2];
                        const double nl = fma(c.x, vr[k2].y, -c.y * vr[k2].x);
                        if (h == 0) w[k2].x = nl; else w[k2].y = nl;
                    }
                }
                Dft<8, -1>::run(w);
                cplx* tile0 = Z + pair2 * PS + k1y * 9;
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) {
                    cplx tq = twy[k1y * 9 + k2];
                    tile0[k2] = (k2 == 0) ? w[0] : cmul(w[k2], tq.x, -tq.y);
                }
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
                    const int ccp = kyi, ccm = kyi ? W2 - kyi : 0;
#pragma unroll
                    for (int n2 = 0; n2 < 4; ++n2) {
                        const cplx* Pr = Z + (n1 + AX * n2) * PS;
                        const cplx pp = Pr[ccp], pm = Pr[ccm];
                        xx[j][n2] = cmake(pp.x + pm.x, pp.y - pm.y);
                        xx[j][n2 + 4] = cmake(pp.y + pm.y, pm.x - pp.x);
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
                    Dft<8, -1>::run(xx[j]);
#pragma unroll
                    for (int k2 = 0; k2 < 8; ++k2) {
                        const int e = 8 * n1 + ((k2 + n1) & 7);
                        cplx tq = twx[n1 * 9 + k2];
                        Z[(e % NPAIR) * PS + ((e / NPAIR) ? s1 : s0)] =
                            (k2 == 0) ? xx[j][0] : cmul(xx[j][k2], tq.x, -tq.y);
                    }
                }
            }
            __syncwarp(FULL);
            {
                const int col = lane >> 3, k2 = lane & 7;
                const int kyi = 4 * u + col;
                const int s0 = kyi, s1 = kyi ? W2 - kyi : NKY0;
                cplx* Rcol = Rb + (size_t)kyi * NX0;
                cplx r0[AX1], r1[AX1];
#pragma unroll
                for (int c = 0; c < AX1; ++c) {  // rhs requested before the butterfly
                    r0[c] = Rcol[k2 + 8 * c];
                    r1[c] = Rcol[k2 + 8 * c + M];
                }
                cplx in[AX];
#pragma unroll
                for (int n1 = 0; n1 < AX; ++n1) {
                    const int e = 8 * n1 + ((k2 + n1) & 7);
                    in[n1] = Z[(e % NPAIR) * PS + ((e / NPAIR) ? s1 : s0)];
                }
                cplx lo[AX1], hi[AX1];
                dft_pruned_out<AX, -1>(in, lo, hi);
#pragma unroll
                for (int c = 0; c < AX1; ++c) {
                    const int i = k2 + 8 * c;
                    Rcol[i] = cmake(fma(coef, lo[c].x, r0[c].x), fma(coef, lo[c].y, r0[c].y));
                    if (i != 0)  // i + M == M is the Nyquist row: untouched
                        Rcol[i + M] = cmake(fma(coef, hi[c].x, r1[c].x), fma(coef, hi[c].y, r1[c].y));
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace gnl
