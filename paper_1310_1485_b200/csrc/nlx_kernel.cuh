// nlx_kernel.cuh -- the x-GLOBAL E x B nonlinearity, the operator the paper ran and timed:
// spectral in y only, real space in x.  PAPER.md:61: "the fields are preprocessed (transposition, extension in y
// direction for dealiasing according to the 3/2-rule) ..., and a fast Fourier transform to real space is applied.
// After multiplication the result is transformed back to the spectral representation, the additional modes are
// deleted, the array is transposed and multiplied with a prefactor, and is finally added to the right-hand side
// vector."  PAPER.md:67: inputs are the x and y components of the E x B velocity and the x and y derivatives of the
// distribution function, plus the right-hand side (5 planes in, 1 out; intensity 1/6).
//
//   per plane, per x:  N(x,y) = vex*dxg + vey*dyg on the padded real grid Ny = 3 nky0,
//                      rhs[x,j] += scale * pref[x] * N^(x,j),  j < nky0.
//
// The paper's seven kernels (Table 3: two transposes, extend, cuFFT x2, multiply, shrink, prefactor) are ONE kernel
// here, bound by HBM (6 planes of traffic per plane, ~2 flop/B):
//   * a CTA takes XT = 16 consecutive x of one plane: every global access is a 256 B run along x (the "transposes"
//     are the index map of the shared-memory staging tile);
//   * the two real fields of a pair travel as ONE complex field (vex + i vey, dxg + i dyg): one complex y-synthesis
//     of length Ny gives both; its non-zero inputs are cc in [0,nky0) (+ky) and (2nky0,3nky0) (-ky, conjugates), so
//     the first radix-A stage is pruned (3/2 rule: "extension" costs no memory and 2/3 of a radix-3 step);
//   * rows r and r+XT/2 of the tile share ONE forward transform (W = N_r + i N_r'); the two are separated in the
//     epilogue, which also deletes the padded modes, applies the prefactor and adds to rhs.
// Twiddles: the Y1 ones (fixed n2 per thread) sit in registers for the life of the persistent CTA, and so do the Y2
// ones when a thread has at most one Y2 item per tile (fixed k1); otherwise they come from the global table through L1
// (a shared-memory table measured slower).  No cuFFT.
#pragma once
#include <cuda_runtime.h>

#include "nl_kernels.cuh"

namespace gnl {

// 16-byte asynchronous copy global -> shared (LDGSTS); `ok` false writes zeros instead (ragged x tail)
__device__ __forceinline__ void cp_async16(cplx* dst_smem, const cplx* src, bool ok)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    const int n = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int NY, int A, int B, int NT, int XT_ = 32>
struct XGlobal {
    static constexpr int XT = XT_, HP = XT / 2;           // x points (rows) and row pairs per tile
    static constexpr int NKY0 = NY / 3, W2 = 2 * NKY0;
    static constexpr int SP = XT + 1;                     // padded row of the staging tile S[field][ky][x]
    static constexpr int S_CPLX = 4 * NKY0 * SP;
    static constexpr int FLAT = Tile<A, B>::FLAT;         // exchange tile of one row: [A][BP]
    static constexpr int E_CPLX = 2 * XT * FLAT;          // (pack, row)
    static constexpr int PP = W2 + 1;                     // padded row of P[pair][cc]; P lives over the pack-1 tiles of E
    static_assert(HP * PP <= XT * FLAT, "P fits over the tiles of the second pack");
    static_assert(NT % XT == 0 && (4 * NKY0) % (NT / XT) == 0 && NKY0 % (NT / XT) == 0, "staging / epilogue split over the threads");
    static constexpr size_t SMEM_BYTES = sizeof(cplx) * (size_t)(S_CPLX + E_CPLX);
};

// grid-stride over tiles; tile t -> plane t / xtiles, x0 = 32 * (t % xtiles).  Software pipeline per CTA: the inputs
// of tile t+1 are copied asynchronously into S (free once Y1 of tile t has consumed it) while Y2, Y3 and the epilogue
// of tile t run; the rhs values of tile t are requested before Y2 and used after Y3.
template <int NY, int A, int B, int NT, int XT_ = 32>
__global__ void __launch_bounds__(NT)
k_xglobal(const cplx* __restrict__ vex, const cplx* __restrict__ vey, const cplx* __restrict__ dxg,
          const cplx* __restrict__ dyg, const double* __restrict__ pref, cplx* __restrict__ rhs,
          const cplx* __restrict__ tw_g, int nx, int xtiles, long long ntiles, double coef)
{
    using C = XGlobal<NY, A, B, NT, XT_>;
    constexpr int XT = C::XT, HP = C::HP, NKY0 = C::NKY0, W2 = C::W2, SP = C::SP, FLAT = C::FLAT, PP = C::PP;
    constexpr int A1 = A / 3, BP = Tile<A, B>::BP, NWARP = NT / XT;  // "warp" = group of XT threads running over x
    constexpr int NEP = NKY0 / NWARP;      // ky rows per group of XT threads (staging of each field, epilogue)
    extern __shared__ cplx smem[];
    cplx* S = smem;
    cplx* E = smem + C::S_CPLX;
    cplx* Pq = E + XT * FLAT;  // over the pack-1 tiles, dead once Y2 has run
    const int lane = threadIdx.x % XT, warp = threadIdx.x / XT;

    // stage the 4 input tiles of tile t: S[f][j][r] = F_f[x0 + r + nx j]; lanes over x (transposition = index map)
    auto stage = [&](long long t) {
        const long long p = t / xtiles;
        const int x0 = (int)(t % xtiles) * XT;
        const size_t base = (size_t)p * (size_t)nx * NKY0 + x0 + lane;
        const bool ok = x0 + lane < nx;
#pragma unroll
        for (int f = 0; f < 4; ++f) {              // the field is a compile-time index: no pointer selects per copy
            const cplx* F = f == 0 ? vex : f == 1 ? vey : f == 2 ? dxg : dyg;
#pragma unroll
            for (int i = 0; i < NEP; ++i) {
                const int j = warp + NWARP * i;
                cp_async16(S + (f * NKY0 + j) * SP + lane, ok ? F + base + (size_t)nx * j : F, ok);
            }
        }
    };

    // Y1 twiddles W_Ny^{k1 n2}: n2 = item % B is the same for every Y1 item of a thread (NT is a multiple of B)
    static_assert(NT % B == 0, "a thread keeps its n2 over the Y1 items");
    cplx tw1[A];
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) tw1[k1] = TWD_G(k1, threadIdx.x % B);

    // Y2 twiddles W_Ny^{k1 k2}: with at most one Y2 item per thread (HP * A <= NT) k1 = threadIdx.x % A is fixed too
    constexpr bool TW2_REGS = (HP * A <= NT);
    [[maybe_unused]] cplx tw2[B];
    if constexpr (TW2_REGS) {
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) tw2[k2] = TWD_G(threadIdx.x % A, k2);
    }

    long long t = blockIdx.x;
    if (t < ntiles) stage(t);
    for (; t < ntiles; t += gridDim.x) {
        const long long p = t / xtiles;
        const int x0 = (int)(t % xtiles) * XT;
        const size_t base = (size_t)p * (size_t)nx * NKY0 + x0;
        cp_async_wait_all();
        __syncthreads();  // S holds tile t; everybody is done with E / P of the previous tile

        // ---- Y1: extension (3/2 rule) + pruned radix-A + twiddle; item = (pack, row, n2) ----
        for (int item = threadIdx.x; item < 2 * XT * B; item += NT) {
            const int n2 = item % B, pr = item / B;  // pr = pack * XT + row
            const int r = pr % XT, pk = pr / XT;
            const cplx* S1 = S + (2 * pk) * NKY0 * SP + r;   // vex | dxg
            const cplx* S2 = S1 + NKY0 * SP;                 // vey | dyg
            cplx lo[A1], hi[A1];
#pragma unroll
            for (int a = 0; a < A1; ++a) {
                const int j = n2 + B * a;                    // +ky: F1 + i F2
                cplx f1 = S1[j * SP], f2 = S2[j * SP];
                if (j == 0) { f1.y = 0.0; f2.y = 0.0; }      // real fields: Im of the ky = 0 mode is ignored
                lo[a] = cmake(f1.x - f2.y, f1.y + f2.x);
                const int jm = NKY0 - j;                     // -ky' at cc = j + nky0: conj F1 + i conj F2; ky' = nky0: none
                const int jc = jm == NKY0 ? 0 : jm;
                const cplx g1 = S1[jc * SP], g2 = S2[jc * SP];
                hi[a] = jm == NKY0 ? cmake(0.0, 0.0) : cmake(g1.x + g2.y, g2.x - g1.y);
            }
            cplx out[A];
            dft_pruned_in<A, +1>(lo, hi, out);
            cplx* Er = E + pr * FLAT + n2;
#pragma unroll
            for (int k1 = 0; k1 < A; ++k1) Er[k1 * BP] = (k1 == 0) ? out[0] : cmul(out[k1], tw1[k1].x, tw1[k1].y);
        }
        __syncthreads();

        // S is free: start copying the next tile; request this tile's rhs values (used after Y3)
        if (t + gridDim.x < ntiles) stage(t + gridDim.x);
        cplx rv[NEP];
        const bool okx = x0 + lane < nx;
#pragma unroll
        for (int i = 0; i < NEP; ++i)
            rv[i] = okx ? rhs[base + lane + (size_t)nx * (warp + NWARP * i)] : cmake(0.0, 0.0);
        const double cpre = okx ? coef * __ldg(pref + x0 + lane) : 0.0;

        // ---- Y2: to real space (both packs, both rows of a pair), multiply, back; item = (pair, k1) ----
        for (int item = threadIdx.x; item < HP * A; item += NT) {
            const int k1 = item % A, q = item / A;
            cplx w[B];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = q + h * HP;
                cplx v1[B], v2[B];
                const cplx* E1 = E + r * FLAT + k1 * BP;
                const cplx* E2 = E1 + XT * FLAT;
#pragma unroll
                for (int n2 = 0; n2 < B; ++n2) { v1[n2] = E1[n2]; v2[n2] = E2[n2]; }
                Dft<B, +1>::run(v1);  // (vex, vey)(x_r, y = k1 + A k2)
                Dft<B, +1>::run(v2);  // (dxg, dyg)
#pragma unroll
                for (int k2 = 0; k2 < B; ++k2) {
                    const double nl = fma(v1[k2].x, v2[k2].x, v1[k2].y * v2[k2].y);  // vex dxg + vey dyg
                    if (h == 0) w[k2].x = nl; else w[k2].y = nl;
                }
            }
            Dft<B, -1>::run(w);
            cplx* Eo = E + q * FLAT + k1 * BP;  // over the slots this item has just read
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                cplx tq;
                if constexpr (TW2_REGS) tq = tw2[k2]; else tq = TWD_G(k1, k2);
                Eo[k2] = (k2 == 0) ? w[0] : cmul(w[k2], tq.x, -tq.y);
            }
        }
        __syncthreads();

        // ---- Y3: pruned-output radix-A ("additional modes are deleted"); item = (pair, k2) -> P[pair][cc] ----
        for (int item = threadIdx.x; item < HP * B; item += NT) {
            const int k2 = item % B, q = item / B;
            cplx in[A];
            const cplx* Er = E + q * FLAT + k2;
#pragma unroll
            for (int n1 = 0; n1 < A; ++n1) in[n1] = Er[n1 * BP];
            cplx lo[A1], hi[A1];
            dft_pruned_out<A, -1>(in, lo, hi);
            cplx* Pr = Pq + q * PP + k2;
#pragma unroll
            for (int c = 0; c < A1; ++c) {
                Pr[B * c] = lo[c];
                Pr[B * c + NKY0] = hi[c];
            }
        }
        __syncthreads();

        // ---- epilogue: separate the two rows of a pair, prefactor, add to rhs; lanes over x ----
        if (okx) {
            const int q = lane % HP;
#pragma unroll
            for (int i = 0; i < NEP; ++i) {
                const int j = warp + NWARP * i;
                const cplx pp = Pq[q * PP + j], pm = Pq[q * PP + (j ? W2 - j : 0)];
                // row q: (P+ + conj P-)/2 ; row q + HP: -i (P+ - conj P-)/2   (the 1/2 and 1/Ny are in coef)
                const cplx n = (lane < HP) ? cmake(pp.x + pm.x, pp.y - pm.y) : cmake(pp.y + pm.y, pm.x - pp.x);
                rhs[base + lane + (size_t)nx * j] = cmake(fma(cpre, n.x, rv[i].x), fma(cpre, n.y, rv[i].y));
            }
        }
    }
}

}  // namespace gnl
