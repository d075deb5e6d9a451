// nl_pipe.cuh -- software-pipelined, persistent versions of the x kernels of the batched path (same steps, same
// scratch layouts as nl_kernels.cuh: SURVEY.md 8(a) A1/A2/A3 and A5/A6).  ncu of the first-generation
// kernels: k_xinv and k_xfwd wait for their global loads (long_scoreboard 3.3 / 5.9 cycles per issued instruction, FP64
// pipe 28 % / 23 %).  Here a CTA stays resident, walks its tiles grid-stride and copies the NEXT tile's inputs into
// shared memory with cp.async (LDGSTS) while the second stage of the current tile runs and its stores drain.
#pragma once
#include <cuda_runtime.h>

#include "nl_kernels.cuh"

namespace gnl {

// 16-byte asynchronous copy global -> shared (LDGSTS, through L2 only)
__device__ __forceinline__ void cp_async_16(cplx* dst_smem, const cplx* src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------------------------
// k_xinv_p: spectral plane F[ky][i] -> Z[bl][m][cc]; tile = CK stored columns of one plane = one CONTIGUOUS block of
// CK * NX0 values of the source, staged in SG.  smem: tw | E (2 CK exchange tiles) | SG.
// ------------------------------------------------------------------------------------------------------------------
template <int NX, int A, int B, int CK, int NT>
struct XInvP {
    static constexpr int NX0 = 2 * (NX / 3);
    static constexpr int TW = A * Tile<A, B>::BP, E_CPLX = 2 * CK * Tile<A, B>::STRIDE, SG_CPLX = CK * NX0;
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)(TW + E_CPLX + SG_CPLX);
    static_assert(SG_CPLX % NT == 0, "the staged block splits evenly over the threads");
};

// ZT: Z is stored TRANSPOSED, Zt[bl][cc][m]: the 8 consecutive m of a warp's stage-2 items form a 128 B run, where the
// row-major store scatters 64 B pieces 2 KB apart (measured: the store pattern costs 29 % of the kernel at Nx = 384).
// k_ybracket_t reads that layout.
template <int NX, int A, int B, int CK, int NT, bool ZT = false>
__global__ void __launch_bounds__(NT)
k_xinv_p(const cplx* __restrict__ src, cplx* __restrict__ Z, const cplx* __restrict__ tw_g,
         int nky0, int nzb, long long vstride, double kxmin, double kymin, int ntot)
{
    using C = XInvP<NX, A, B, CK, NT>;
    static_assert(A * B == NX && A % 3 == 0, "NX = A*B with 3 | A");
    constexpr int A1 = A / 3, M = NX / 3, NX0 = 2 * M;
    constexpr int BP = Tile<A, B>::BP, CS = Tile<A, B>::STRIDE, NCP = C::SG_CPLX / NT;
    extern __shared__ cplx smem[];
    cplx* tw = smem;
    cplx* E = smem + C::TW;
    cplx* SG = E + C::E_CPLX;
    const int ntile = nky0 / CK;
    const int W2 = 2 * nky0;

    auto stage = [&](int t) {
        const int bl = t / ntile, ky0 = (t % ntile) * CK;
        const cplx* F = src + ((size_t)(bl % nzb) + (size_t)vstride * (bl / nzb)) * ((size_t)NX0 * nky0) + (size_t)ky0 * NX0;
#pragma unroll
        for (int i = 0; i < NCP; ++i) cp_async_16(SG + threadIdx.x + NT * i, F + threadIdx.x + NT * i);
    };

    int t = blockIdx.x;
    if (t < ntot) stage(t);
    load_twiddles_ab<A, B>(tw, tw_g);
    for (; t < ntot; t += gridDim.x) {
        const int bl = t / ntile, ky0 = (t % ntile) * CK;
        cplx* Zb = Z + (size_t)bl * NX * W2;
        cp_async_wait();
        __syncthreads();  // SG holds tile t (and tw is loaded); stage 2 of the previous tile has read E

        // stage 1: derivative, pad, pruned radix-A over n1 for fixed n2 (n = n2 + B*n1), twiddle W_NX^{n2 k1}
        for (int item = threadIdx.x; item < 2 * CK * B; item += NT) {
            const int n2 = item % B, c2 = item / B;
            const int col = c2 % CK, sg = c2 / CK;
            const int kyi = ky0 + col;
            if (sg == 1 && kyi == 0) continue;  // there is no -0 column
            const cplx* Fc = SG + col * NX0;
            const double ky = kymin * (double)kyi;
            const double kys = sg ? ky : -ky;  // (i kx - ky) F for +ky, (i kx + ky) F for -ky
            cplx lo[A1], hi[A1];
#pragma unroll
            for (int a = 0; a < A1; ++a) {
                {
                    const int i = n2 + B * a;  // kx >= 0 rows
                    const double kx = kxmin * (double)i;
                    cplx f = Fc[i];
                    if (kyi == 0) {  // Hermitian part of the ky = 0 column (R7)
                        cplx fm = Fc[(NX0 - i) % NX0];
                        f = cmake(0.5 * (f.x + fm.x), 0.5 * (f.y - fm.y));
                    }
                    lo[a] = cmake(fma(kys, f.x, -kx * f.y), fma(kx, f.x, kys * f.y));
                }
                {
                    const int i = n2 + B * a + M;  // kx < 0 rows, i in [M, 2M); i == M is the Nyquist row
                    const double kx = kxmin * (double)(i - NX0);
                    cplx f = Fc[i];
                    if (kyi == 0) {
                        cplx fm = Fc[NX0 - i];
                        f = cmake(0.5 * (f.x + fm.x), 0.5 * (f.y - fm.y));
                    }
                    cplx v = cmake(fma(kys, f.x, -kx * f.y), fma(kx, f.x, kys * f.y));
                    hi[a] = (i == M) ? cmake(0.0, 0.0) : v;
                }
            }
            cplx out[A];
            dft_pruned_in<A, +1>(lo, hi, out);
            cplx* Ec = E + c2 * CS + n2;
#pragma unroll
            for (int k1 = 0; k1 < A; ++k1) {
                cplx w = TWD(k1, n2);
                Ec[k1 * BP] = (k1 == 0) ? out[0] : cmul(out[k1], w.x, w.y);
            }
        }
        __syncthreads();
        if (t + (int)gridDim.x < ntot) stage(t + gridDim.x);  // SG is free: fetch the next tile behind stage 2

        // stage 2: radix-B over n2 for fixed k1; output m = k1 + A*k2
        for (int item = threadIdx.x; item < 2 * CK * A; item += NT) {
            const int col = item % CK, rest = item / CK;
            const int k1 = rest % A, sg = rest / A;
            const int c2 = sg * CK + col, kyi = ky0 + col;
            const bool zero = (sg == 1 && kyi == 0);
            cplx v[B];
            const cplx* Ec = E + c2 * CS + k1 * BP;
#pragma unroll
            for (int n2 = 0; n2 < B; ++n2) v[n2] = zero ? cmake(0.0, 0.0) : Ec[n2];
            Dft<B, +1>::run(v);
            const int cc = sg ? (kyi ? W2 - kyi : nky0) : kyi;
            cplx* Zc = Zb + cc;
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                const int m = k1 + A * k2;
                if constexpr (ZT) Zb[(size_t)cc * NX + m] = sg ? cconj(v[k2]) : v[k2];
                else Zc[(size_t)m * W2] = sg ? cconj(v[k2]) : v[k2];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// k_ybracket_t: as k_ybracket (chi shared over v), reading the g side from the TRANSPOSED Zt[bl][cc][m].  A tile is 8
// row pairs (m0..m0+7 and m0+Nx/2..+7): in Y1 the lanes run over the 16 rows, so every load is two 128 B runs.
// smem: 16 exchange tiles with an odd row stride (lanes over rows stay bank-conflict free).  grid as k_ybracket, RP = 8.
// ------------------------------------------------------------------------------------------------------------------
template <int NY, int A, int B, int NT, int RP_ = 8>
struct YBracketT {
    static constexpr int RP = RP_, RSP = odd_up(Tile<A, B>::FLAT);
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)(2 * RP * RSP);
};

template <int NY, int A, int B, int NT, int RP_ = 8>
__global__ void __launch_bounds__(NT)
k_ybracket_t(const cplx* __restrict__ Zt, const cplx* __restrict__ R, cplx* __restrict__ P,
             const cplx* __restrict__ tw_g, int Nx, int nzb, int vfast)
{
    constexpr int RP = RP_, A1 = A / 3, NKY0 = NY / 3, W2 = 2 * NKY0;
    constexpr int BP = Tile<A, B>::BP, RS = YBracketT<NY, A, B, NT, RP_>::RSP;
    extern __shared__ cplx smem[];
    cplx* E = smem;
    const int half = Nx / 2;
    const int ntile = half / RP;
    int bl, m0;
    if (vfast) {
        const int nvc = gridDim.x / (ntile * nzb);
        m0 = ((blockIdx.x / nvc) % ntile) * RP;
        bl = blockIdx.x / (nvc * ntile) + nzb * (blockIdx.x % nvc);
    } else {
        bl = blockIdx.x / ntile;
        m0 = (blockIdx.x % ntile) * RP;
    }
    const int ql = bl % nzb;
    const cplx* Zp = Zt + (size_t)bl * Nx * W2;

    // Y1: pruned radix-A + twiddle; item = (row r of 16, n2), lanes over the rows
    for (int item = threadIdx.x; item < 2 * RP * B; item += NT) {
        const int r = item % (2 * RP), n2 = item / (2 * RP);
        const int m = m0 + (r % RP) + (r / RP) * half;
        cplx lo[A1], hi[A1];
#pragma unroll
        for (int a = 0; a < A1; ++a) {
            lo[a] = __ldg(reinterpret_cast<const double2*>(Zp + (size_t)(n2 + B * a) * Nx + m));
            hi[a] = __ldg(reinterpret_cast<const double2*>(Zp + (size_t)(n2 + B * a + NKY0) * Nx + m));
        }
        cplx out[A];
        dft_pruned_in<A, +1>(lo, hi, out);
        cplx* Er = E + r * RS + n2;
#pragma unroll
        for (int k1 = 0; k1 < A; ++k1) {
            const cplx w = TWD_G(k1, n2);
            Er[k1 * BP] = (k1 == 0) ? out[0] : cmul(out[k1], w.x, w.y);
        }
    }
    __syncthreads();

    // Y2: radix-B to real space for both rows of a pair, bracket, radix-B back + twiddle (in place)
    for (int item = threadIdx.x; item < RP * A; item += NT) {
        const int k1 = item % A, r = item / A;
        cplx w[B];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int row = r + h * RP;
            const int m = m0 + r + h * half;
            cplx v[B];
            const cplx* Er = E + row * RS + k1 * BP;
#pragma unroll
            for (int n2 = 0; n2 < B; ++n2) v[n2] = Er[n2];
            Dft<B, +1>::run(v);
            const cplx* Rc = R + ((size_t)ql * Nx + m) * NY + k1;
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                const cplx c = Rc[A * k2];  // (dx chi, dy chi)
                const double nl = fma(c.x, v[k2].y, -c.y * v[k2].x);
                if (h == 0) w[k2].x = nl; else w[k2].y = nl;
            }
        }
        Dft<B, -1>::run(w);
        cplx* Er = E + r * RS + k1 * BP;
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            cplx tq = TWD_G(k1, k2);
            Er[k2] = (k2 == 0) ? w[0] : cmul(w[k2], tq.x, -tq.y);
        }
    }
    __syncthreads();

    // Y3: pruned-output radix-A over n1 for fixed k2; j = k2 + B*k1
    for (int item = threadIdx.x; item < RP * B; item += NT) {
        const int k2 = item % B, r = item / B;
        cplx in[A];
        const cplx* Er = E + r * RS + k2;
#pragma unroll
        for (int n1 = 0; n1 < A; ++n1) in[n1] = Er[n1 * BP];
        cplx lo[A1], hi[A1];
        dft_pruned_out<A, -1>(in, lo, hi);
        cplx* Pp = P + ((size_t)bl * half + m0 + r) * W2 + k2;
#pragma unroll
        for (int cq = 0; cq < A1; ++cq) {
            Pp[B * cq] = lo[cq];
            Pp[B * cq + NKY0] = hi[cq];
        }
    }
}

}  // namespace gnl
