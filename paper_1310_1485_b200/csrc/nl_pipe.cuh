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

template <int NX, int A, int B, int CK, int NT>
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
                Zc[(size_t)m * W2] = sg ? cconj(v[k2]) : v[k2];
            }
        }
    }
}

}  // namespace gnl
