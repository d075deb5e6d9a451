// nl_kernels.cuh -- the sm_100a kernels of the E x B nonlinearity (batched, scratch in L2).
//
// Hot path:
//   k_xinv      A1 derivative + A2 zero-pad + x half of A3 (to real space), for g and for chi
//   k_yreal     y half of A3 for chi: real-space (dx chi, dy chi), shared by the nv planes
//   k_ybracket  y half of A3 for g + A4 bracket + y half of A5 (back to spectral)
//   k_xfwd      x half of A5 + A6 delete modes, prefactor, add to rhs
//
// Data flow per plane (N = Nx or Ny is split as A*B, A a multiple of 3 carrying the 3/2 pruning):
//   * the two real fields (dx f, dy f) of one source are carried as ONE complex field dx f + i dy f.
//     Its spectrum at (kx,+ky) is (i kx - ky) F(kx,ky); at (kx,-ky) it is the conjugate of the
//     x-synthesis of (i kx + ky) F(kx,ky).  k_xinv therefore runs two x-FFTs per stored column and
//     writes Z[plane][m][cc], cc in [0, 2 nky0): cc = ky for ky >= 0, cc = 2 nky0 - ky for -ky.
//     These are exactly the non-zero inputs of the padded complex y-FFT of length Ny = 3 nky0.
//   * k_ybracket pairs the rows m and m + Nx/2: W = N_m + i N_m' goes through ONE forward y-FFT;
//     P[plane][m][cc] keeps both halves (+ky, -ky) of its spectrum and k_xfwd separates the two rows
//     while loading, N^_m = (P+ + conj P-)/2, N^_m' = (P+ - conj P-)/(2i).
// Scratch Z, P, Rchi is sized per batch of planes so that it stays resident in the 126 MB L2.
#pragma once
#include <cuda_runtime.h>

#include "dft_regs.cuh"

// Twiddle W_N^{i j} of a two-stage transform.  The x kernels read it from a padded shared-memory table filled in the
// CTA prologue; the y kernels read the global table through L1 (no prologue, no barrier before the first row load):
// measured on B200, that is faster for k_yreal / k_ybracket (-16 % at 144x144) and slower for k_xinv / k_xfwd.
#define TWD(i, j) tw[(i) * BP + (j)]
#define TWD_G(i, j) __ldg(reinterpret_cast<const double2*>(tw_g) + (i) * (j))

namespace gnl {

__host__ __device__ constexpr int odd_up(int v) { return v | 1; }

// shared-memory exchange tile of one length-N FFT: [A][BP] complex, BP odd, block stride odd
template <int A, int B>
struct Tile {
    static constexpr int BP = odd_up(B);
    static constexpr int STRIDE = odd_up(A * BP);  // x kernels: lanes run over columns (stride must be odd)
    static constexpr int FLAT = A * BP;            // y kernels: lanes run over (row, k1) as one flat index
};

// Twiddle table of one length N = A*B in shared memory, laid out [k1][n2] with row stride BP (odd):
// T[k1*BP + n2] = W_N^{n2 k1}.  Conflict-free both for lanes over n2 and for lanes over k1.
template <int A, int B>
__device__ __forceinline__ void load_twiddles_ab(cplx* tw_s, const cplx* __restrict__ tw_g)
{
    constexpr int BP = Tile<A, B>::BP;
    for (int t = threadIdx.x; t < A * B; t += blockDim.x) {
        const int k1 = t / B, n2 = t % B;
        tw_s[k1 * BP + n2] = tw_g[k1 * n2];
    }
}

// ------------------------------------------------------------------------------------------------
// k_xinv: spectral plane F[ky][i]  ->  Z[bl][m][cc]   (x-synthesis of (i kx -+ ky) F, padded 3/2)
// grid = planes_in_batch * (nky0 / CK); one CTA does CK stored columns = 2 CK FFTs of length NX.
// ------------------------------------------------------------------------------------------------
// SEQ: the +ky and the -ky transforms of the CK columns go through E one after the other, so E holds CK tiles
// instead of 2*CK and twice as many columns fit (128 B instead of 64 B pieces in the row-major store of Z).
template <int NX, int A, int B, int CK, int NT, bool SEQ = false>
__global__ void __launch_bounds__(NT)
k_xinv(const cplx* __restrict__ src, cplx* __restrict__ Z, const cplx* __restrict__ tw_g,
       int nky0, int nzb, long long vstride, double kxmin, double kymin)
{
    static_assert(A * B == NX && A % 3 == 0, "NX = A*B with 3 | A");
    constexpr int A1 = A / 3, M = NX / 3, NX0 = 2 * M;
    constexpr int BP = Tile<A, B>::BP, CS = Tile<A, B>::STRIDE;
    extern __shared__ cplx smem[];
    cplx* tw = smem;
    cplx* E = smem + A * BP;

    const int ntile = nky0 / CK;
    const int bl = blockIdx.x / ntile;
    const int ky0 = (blockIdx.x % ntile) * CK;
    const int W2 = 2 * nky0;
    const cplx* F = src + ((size_t)(bl % nzb) + (size_t)vstride * (bl / nzb)) * ((size_t)NX0 * nky0);
    cplx* Zb = Z + (size_t)bl * NX * W2;

    load_twiddles_ab<A, B>(tw, tw_g);
    __syncthreads();
    constexpr int NSG = SEQ ? 1 : 2;  // signs per pass through E

#pragma unroll 1
    for (int sg0 = 0; sg0 < 2; sg0 += NSG) {
    // stage 1: pruned radix-A over n1 for fixed n2 (n = n2 + B*n1), then twiddle W_NX^{n2 k1}
    for (int item = threadIdx.x; item < NSG * CK * B; item += NT) {
        const int n2 = item % B, c2 = item / B;
        const int col = c2 % CK, sg = sg0 + c2 / CK;
        const int kyi = ky0 + col;
        if (sg == 1 && kyi == 0) continue;  // there is no -0 column
        const cplx* Fc = F + (size_t)kyi * NX0;
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

    // stage 2: radix-B over n2 for fixed k1; output m = k1 + A*k2
    for (int item = threadIdx.x; item < NSG * CK * A; item += NT) {
        const int col = item % CK, rest = item / CK;
        const int k1 = rest % A, sg = sg0 + rest / A;
        const int c2 = (rest / A) * CK + col, kyi = ky0 + col;
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
    if (SEQ && sg0 == 0) __syncthreads();  // stage 2 has read E before the -ky pass overwrites it
    }
}

// ------------------------------------------------------------------------------------------------
// stage 1 of the y-synthesis, shared by k_yreal and k_ybracket: rows of Z -> exchange tile
// ------------------------------------------------------------------------------------------------
template <int NY, int A, int B>
__device__ __forceinline__ void y_stage1(const cplx* __restrict__ Zr, const cplx* __restrict__ tw_g, cplx* Er, int n2)
{
    constexpr int A1 = A / 3, NKY0 = NY / 3, BP = Tile<A, B>::BP;
    cplx lo[A1], hi[A1];
#pragma unroll
    for (int a = 0; a < A1; ++a) {
        lo[a] = Zr[n2 + B * a];          // j = n2 + B*a            in [0, nky0)
        hi[a] = Zr[n2 + B * a + NKY0];   // j = n2 + B*(a + 2 A1)   in [2 nky0, 3 nky0), cc = j - nky0
    }
    cplx out[A];
    dft_pruned_in<A, +1>(lo, hi, out);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) {
        cplx w = TWD_G(k1, n2);
        Er[k1 * BP + n2] = (k1 == 0) ? out[0] : cmul(out[k1], w.x, w.y);
    }
}

// ------------------------------------------------------------------------------------------------
// k_yreal: Z[ql][m][cc] -> R[ql][m][y] = (dx chi, dy chi)(m, y).  grid = chi_planes * (Nx / RT).
// ------------------------------------------------------------------------------------------------
template <int NY, int A, int B, int RT, int NT>
__global__ void __launch_bounds__(NT)
k_yreal(const cplx* __restrict__ Z, cplx* __restrict__ R, const cplx* __restrict__ tw_g, int Nx)
{
    constexpr int W2 = 2 * (NY / 3);
    constexpr int BP = Tile<A, B>::BP, RS = Tile<A, B>::FLAT;
    extern __shared__ cplx smem[];
    cplx* E = smem;
    const int ntile = Nx / RT;
    const int ql = blockIdx.x / ntile;
    const int m0 = (blockIdx.x % ntile) * RT;
    for (int item = threadIdx.x; item < RT * B; item += NT) {
        const int n2 = item % B, r = item / B;
        y_stage1<NY, A, B>(Z + ((size_t)ql * Nx + m0 + r) * W2, tw_g, E + r * RS, n2);
    }
    __syncthreads();
    for (int item = threadIdx.x; item < RT * A; item += NT) {
        const int k1 = item % A, r = item / A;
        cplx v[B];
        const cplx* Er = E + r * RS + k1 * BP;
#pragma unroll
        for (int n2 = 0; n2 < B; ++n2) v[n2] = Er[n2];
        Dft<B, +1>::run(v);
        cplx* Rr = R + ((size_t)ql * Nx + m0 + r) * NY + k1;
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) Rr[A * k2] = v[k2];
    }
}

// ------------------------------------------------------------------------------------------------
// k_ybracket: Z[bl][m][cc] (g) and R[ql][m][y] (chi) -> P[bl][pair][cc].
// grid = planes_in_batch * (Nx/2 / RP); one CTA does RP row pairs (m, m + Nx/2).
// ------------------------------------------------------------------------------------------------
// EM: chi = phi_bar - v_par * A_par_bar is composed HERE, in real space and by linearity:
// R holds the real-space fields of phi_bar, R2 those of A_par_bar (one plane per z each, shared by all v), and
// vp[bl / nzb] is the v_par coefficient of plane bl.  Per-plane chi is then never stored nor transformed.
template <int NY, int A, int B, int RP, int NT, bool EM = false>
__global__ void __launch_bounds__(NT)
k_ybracket(const cplx* __restrict__ Z, const cplx* __restrict__ R, cplx* __restrict__ P,
           const cplx* __restrict__ tw_g, int Nx, int nzb, int chi_per_plane, int vfast,
           const cplx* __restrict__ R2 = nullptr, const double* __restrict__ vp = nullptr)
{
    constexpr int A1 = A / 3, NKY0 = NY / 3, W2 = 2 * NKY0;
    constexpr int BP = Tile<A, B>::BP, RS = Tile<A, B>::FLAT;
    extern __shared__ cplx smem[];
    cplx* E = smem;
    const int half = Nx / 2;
    const int ntile = half / RP;
    int bl, m0;
    if (vfast) {
        // CTAs numbered v-fastest: neighbours in launch order work on the same rows of the same chi plane (one z,
        // all v of the batch), so chi rows too large to stay in L2 are fetched from HBM once per batch
        const int nvc = gridDim.x / (ntile * nzb);
        m0 = ((blockIdx.x / nvc) % ntile) * RP;
        bl = blockIdx.x / (nvc * ntile) + nzb * (blockIdx.x % nvc);
    } else {
        bl = blockIdx.x / ntile;
        m0 = (blockIdx.x % ntile) * RP;
    }
    const int ql = chi_per_plane ? bl : bl % nzb;

    // Y1: pruned radix-A + twiddle for the 2*RP rows of the tile
    for (int item = threadIdx.x; item < 2 * RP * B; item += NT) {
        const int n2 = item % B, r = item / B;
        const int m = m0 + (r % RP) + (r / RP) * half;
        y_stage1<NY, A, B>(Z + ((size_t)bl * Nx + m) * W2, tw_g, E + r * RS, n2);
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
            Dft<B, +1>::run(v);  // v[k2] = (dx g + i dy g)(m, y = k1 + A*k2)
            const cplx* Rc = R + ((size_t)ql * Nx + m) * NY + k1;
            [[maybe_unused]] const cplx* Rc2 = EM ? R2 + ((size_t)ql * Nx + m) * NY + k1 : nullptr;
            [[maybe_unused]] const double vpar = EM ? __ldg(vp + bl / nzb) : 0.0;
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                cplx c = Rc[A * k2];  // (dx chi, dy chi)
                if constexpr (EM) {
                    const cplx a2 = Rc2[A * k2];  // (dx A_par, dy A_par)
                    c = cmake(fma(-vpar, a2.x, c.x), fma(-vpar, a2.y, c.y));
                }
                const double nl = fma(c.x, v[k2].y, -c.y * v[k2].x);  // dx chi dy g - dy chi dx g
                if (h == 0) w[k2].x = nl; else w[k2].y = nl;
            }
        }
        Dft<B, -1>::run(w);  // n = k1 + A*n2  ->  U[n1 = k1][k2]
        cplx* Er = E + r * RS + k1 * BP;
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            cplx t = TWD_G(k1, k2);
            Er[k2] = (k2 == 0) ? w[0] : cmul(w[k2], t.x, -t.y);
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
        for (int c = 0; c < A1; ++c) {
            Pp[B * c] = lo[c];         // j in [0, nky0)
            Pp[B * c + NKY0] = hi[c];  // j in [2 nky0, 3 nky0), cc = j - nky0
        }
    }
}

// ------------------------------------------------------------------------------------------------
// k_ybracket_cv: chi per plane (chi_has_v = 1).  Z[bl][m][cc] (g) and Zc[bl][m][cc] (chi, the same x-synthesis) ->
// P[bl][pair][cc].  With one chi plane per g plane there is nothing to share across v, so the real-space chi
// fields are NOT written to and read back from HBM (k_yreal + the R reads of k_ybracket: 2 x 4.5 planes of traffic per
// plane, which made both kernels HBM bound at configs[4]): the y-synthesis of the chi rows runs here, next to that
// of the g rows.  smem: 4*RP exchange tiles (g rows, then chi rows).  grid = planes_in_batch * (Nx/2 / RP).
// ------------------------------------------------------------------------------------------------
template <int NY, int A, int B, int RP, int NT>
__global__ void __launch_bounds__(NT)
k_ybracket_cv(const cplx* __restrict__ Z, const cplx* __restrict__ Zc, cplx* __restrict__ P,
              const cplx* __restrict__ tw_g, int Nx)
{
    constexpr int A1 = A / 3, NKY0 = NY / 3, W2 = 2 * NKY0;
    constexpr int BP = Tile<A, B>::BP, RS = Tile<A, B>::FLAT;
    extern __shared__ cplx smem[];
    cplx* E = smem;
    cplx* Ec = smem + 2 * RP * RS;
    const int half = Nx / 2;
    const int ntile = half / RP;
    const int bl = blockIdx.x / ntile;
    const int m0 = (blockIdx.x % ntile) * RP;

    // Y1: pruned radix-A + twiddle for the 2*RP rows of g and the 2*RP rows of chi
    for (int item = threadIdx.x; item < 4 * RP * B; item += NT) {
        const int n2 = item % B, r4 = item / B;
        const int r = r4 % (2 * RP), src = r4 / (2 * RP);
        const int m = m0 + (r % RP) + (r / RP) * half;
        y_stage1<NY, A, B>((src ? Zc : Z) + ((size_t)bl * Nx + m) * W2, tw_g, E + r4 * RS, n2);
    }
    __syncthreads();

    // Y2: both rows of a pair of g and of chi to real space, bracket, radix-B back + twiddle (in place)
    for (int item = threadIdx.x; item < RP * A; item += NT) {
        const int k1 = item % A, r = item / A;
        cplx w[B];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int row = r + h * RP;
            cplx v[B], c[B];
            const cplx* Er = E + row * RS + k1 * BP;
            const cplx* Cr = Ec + row * RS + k1 * BP;
#pragma unroll
            for (int n2 = 0; n2 < B; ++n2) { v[n2] = Er[n2]; c[n2] = Cr[n2]; }
            Dft<B, +1>::run(v);  // (dx g + i dy g)(m, y = k1 + A*k2)
            Dft<B, +1>::run(c);  // (dx chi + i dy chi)
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                const double nl = fma(c[k2].x, v[k2].y, -c[k2].y * v[k2].x);  // dx chi dy g - dy chi dx g
                if (h == 0) w[k2].x = nl; else w[k2].y = nl;
            }
        }
        Dft<B, -1>::run(w);
        cplx* Er = E + r * RS + k1 * BP;
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            cplx t = TWD_G(k1, k2);
            Er[k2] = (k2 == 0) ? w[0] : cmul(w[k2], t.x, -t.y);
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
        for (int c = 0; c < A1; ++c) {
            Pp[B * c] = lo[c];
            Pp[B * c + NKY0] = hi[c];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// k_xfwd: P[bl][pair][cc] -> rhs[ky][i] += coef * X.  grid = planes_in_batch * (nky0 / CK).
// ------------------------------------------------------------------------------------------------
template <int NX, int A, int B, int CK, int NT>
__global__ void __launch_bounds__(NT)
k_xfwd(const cplx* __restrict__ P, cplx* __restrict__ rhs, const cplx* __restrict__ tw_g,
       int nky0, int nzb, long long vstride, double coef)
{
    static_assert(B % 2 == 0, "row pairing m, m + NX/2 needs an even B");
    constexpr int A1 = A / 3, M = NX / 3, NX0 = 2 * M, HALF = NX / 2;
    constexpr int BP = Tile<A, B>::BP, CS = Tile<A, B>::STRIDE;
    extern __shared__ cplx smem[];
    cplx* tw = smem;
    cplx* E = smem + A * BP;
    const int ntile = nky0 / CK;
    const int bl = blockIdx.x / ntile;
    const int ky0 = (blockIdx.x % ntile) * CK;
    const int W2 = 2 * nky0;
    const cplx* Pb = P + (size_t)bl * HALF * W2;
    cplx* Rb = rhs + ((size_t)(bl % nzb) + (size_t)vstride * (bl / nzb)) * ((size_t)NX0 * nky0);
    load_twiddles_ab<A, B>(tw, tw_g);
    __syncthreads();

    // stage 1: unpack the row pair, radix-B over n2 for fixed n1 (m = n1 + A*n2), twiddle W^{-n1 k2}
    for (int item = threadIdx.x; item < CK * A; item += NT) {
        const int col = item % CK, n1 = item / CK;
        const int kyi = ky0 + col;
        const int ccp = kyi, ccm = kyi ? W2 - kyi : 0;
        cplx x[B];
#pragma unroll
        for (int n2 = 0; n2 < B / 2; ++n2) {
            const cplx* Pr = Pb + (size_t)(n1 + A * n2) * W2;
            const cplx pp = Pr[ccp], pm = Pr[ccm];
            x[n2] = cmake(pp.x + pm.x, pp.y - pm.y);           // 2 N^_m      = P+ + conj P-
            x[n2 + B / 2] = cmake(pp.y + pm.y, pm.x - pp.x);   // 2 N^_m'     = -i (P+ - conj P-)
        }
        Dft<B, -1>::run(x);
        cplx* Ec = E + col * CS + n1 * BP;
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            cplx t = TWD(n1, k2);
            Ec[k2] = (k2 == 0) ? x[0] : cmul(x[k2], t.x, -t.y);
        }
    }
    __syncthreads();

    // stage 2: pruned-output radix-A over n1 for fixed k2; k = k2 + B*k1; delete modes, scale, add
    for (int item = threadIdx.x; item < CK * B; item += NT) {
        const int k2 = item % B, col = item / B;
        const int kyi = ky0 + col;
        cplx in[A];
        const cplx* Ec = E + col * CS + k2;
#pragma unroll
        for (int n1 = 0; n1 < A; ++n1) in[n1] = Ec[n1 * BP];
        cplx lo[A1], hi[A1];
        dft_pruned_out<A, -1>(in, lo, hi);
        cplx* Rc = Rb + (size_t)kyi * NX0;
#pragma unroll
        for (int c = 0; c < A1; ++c) {
            const int i = k2 + B * c;  // kx >= 0
            cplx r0 = Rc[i];
            Rc[i] = cmake(fma(coef, lo[c].x, r0.x), fma(coef, lo[c].y, r0.y));
            const int i2 = i + M;  // kx < 0; i2 == M is the Nyquist row: untouched
            if (i2 != M) {
                cplx r1 = Rc[i2];
                Rc[i2] = cmake(fma(coef, hi[c].x, r1.x), fma(coef, hi[c].y, r1.y));
            }
        }
    }
}

}  // namespace gnl
