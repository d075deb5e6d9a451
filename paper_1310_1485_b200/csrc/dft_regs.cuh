// dft_regs.cuh -- register-resident DFT butterflies of small composite radix (2^a 3^b), FP64.
//
// Every index below is a compile-time constant after template expansion, so a cplx[R] array lives in
// registers and permutations are free.  Twiddles of the in-register radices are literals from
// twiddle_consts.cuh; multiplications by 1, -1, +-i are eliminated at compile time.
//
// Sign convention: Dft<R,S> computes X[k] = sum_n x[n] exp(S*2*pi*i*n*k/R), S=+1 synthesis (to real
// space), S=-1 analysis.  Unnormalised.
//
// Pruned variants implement the 3/2-rule structure ("extension ... for dealiasing
// according to the 3/2-rule" / "the additional modes are deleted"): with R = 3*R1 the middle third of
// the inputs is zero on the way to real space (dft_pruned_in) and the middle third of the outputs is
// never needed on the way back (dft_pruned_out), so the radix-3 step loses a third of its work.
#pragma once
#include <type_traits>

#include "twiddle_consts.cuh"

namespace gnl {

typedef double2 cplx;

__device__ __forceinline__ cplx cmake(double x, double y) { return make_double2(x, y); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return cmake(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cconj(cplx a) { return cmake(a.x, -a.y); }
// a * (c + i s)
__device__ __forceinline__ cplx cmul(cplx a, double c, double s)
{
    return cmake(fma(-a.y, s, a.x * c), fma(a.y, c, a.x * s));
}

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F&& f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// v * W_R^(S*J), J compile time
template <int R, int J, int S>
__device__ __forceinline__ cplx mul_w(cplx v)
{
    constexpr int j = ((J % R) + R) % R;
    if constexpr (j == 0) {
        return v;
    } else if constexpr ((4 * j) % R == 0) {
        constexpr int q = (4 * j) / R;  // quarter turns in direction S
        if constexpr (q == 2)
            return cmake(-v.x, -v.y);
        else if constexpr ((q == 1) == (S > 0))
            return cmake(-v.y, v.x);  // * (+i)
        else
            return cmake(v.y, -v.x);  // * (-i)
    } else {
        static_assert(kTwBase % R == 0, "radix must divide the literal twiddle table length");
        constexpr double c = kCos288[j * (kTwBase / R)];
        constexpr double s = (S > 0 ? 1.0 : -1.0) * kSin288[j * (kTwBase / R)];
        return cmul(v, c, s);
    }
}

constexpr double kHalfSqrt3 = 0.8660254037844386467637231707529362;

template <int R, int S>
struct Dft;

template <int S>
struct Dft<1, S> {
    static __device__ __forceinline__ void run(cplx (&)[1]) {}
};

template <int S>
struct Dft<2, S> {
    static __device__ __forceinline__ void run(cplx (&v)[2])
    {
        cplx a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <int S>
struct Dft<3, S> {
    static __device__ __forceinline__ void run(cplx (&v)[3])
    {
        constexpr double h = S * kHalfSqrt3;
        cplx a = v[0], t = cadd(v[1], v[2]), u = csub(v[1], v[2]);
        v[0] = cadd(a, t);
        cplx m = cmake(fma(-0.5, t.x, a.x), fma(-0.5, t.y, a.y));
        v[1] = cmake(fma(-h, u.y, m.x), fma(h, u.x, m.y));  // m + S*i*h*u
        v[2] = cmake(fma(h, u.y, m.x), fma(-h, u.x, m.y));  // m - S*i*h*u
    }
};

template <int S>
struct Dft<4, S> {
    static __device__ __forceinline__ void run(cplx (&v)[4])
    {
        cplx p = cadd(v[0], v[2]), q = csub(v[0], v[2]);
        cplx r = cadd(v[1], v[3]), d = csub(v[1], v[3]);
        cplx id = (S > 0) ? cmake(-d.y, d.x) : cmake(d.y, -d.x);  // S*i*d
        v[0] = cadd(p, r);
        v[2] = csub(p, r);
        v[1] = cadd(q, id);
        v[3] = csub(q, id);
    }
};

// second half of a decimation-in-frequency radix 8: a[n] = x[n] + x[n+4], b[n] = x[n] - x[n+4] -> X[0..7]
template <int S>
__device__ __forceinline__ void dft8_tail(const cplx (&a)[4], const cplx (&b)[4], cplx (&v)[8])
{
    constexpr double r = 0.70710678118654752440084436210484903928;  // 1/sqrt(2)
    {  // even outputs: DFT4 of a
        const cplx p = cadd(a[0], a[2]), q = csub(a[0], a[2]), rr = cadd(a[1], a[3]), d = csub(a[1], a[3]);
        const cplx id = (S > 0) ? cmake(-d.y, d.x) : cmake(d.y, -d.x);  // S i d
        v[0] = cadd(p, rr);
        v[4] = csub(p, rr);
        v[2] = cadd(q, id);
        v[6] = csub(q, id);
    }
    {  // odd outputs: DFT4 of c[n] = b[n] W_8^{S n}; c1 = r u1, c3 = r u3 with the scale applied in the FMAs
        const cplx c2 = (S > 0) ? cmake(-b[2].y, b[2].x) : cmake(b[2].y, -b[2].x);            // b2 (S i)
        const cplx u1 = (S > 0) ? cmake(b[1].x - b[1].y, b[1].x + b[1].y)                      // b1 (1 + S i)
                                : cmake(b[1].x + b[1].y, b[1].y - b[1].x);
        const cplx u3 = (S > 0) ? cmake(-(b[3].x + b[3].y), b[3].x - b[3].y)                   // b3 (-1 + S i)
                                : cmake(b[3].y - b[3].x, -(b[3].x + b[3].y));
        const cplx p = cadd(b[0], c2), q = csub(b[0], c2), s13 = cadd(u1, u3), d13 = csub(u1, u3);
        v[1] = cmake(fma(r, s13.x, p.x), fma(r, s13.y, p.y));
        v[5] = cmake(fma(-r, s13.x, p.x), fma(-r, s13.y, p.y));
        // q +- S i (r d13)
        v[3] = (S > 0) ? cmake(fma(-r, d13.y, q.x), fma(r, d13.x, q.y)) : cmake(fma(r, d13.y, q.x), fma(-r, d13.x, q.y));
        v[7] = (S > 0) ? cmake(fma(r, d13.y, q.x), fma(-r, d13.x, q.y)) : cmake(fma(-r, d13.y, q.x), fma(r, d13.x, q.y));
    }
}

// Radix 8, decimation in frequency, with the 1/sqrt(2) of W_8 and W_8^3 folded into the last layer's FMAs:
// 48 FP64 instructions (32 adds of the two radix-4 halves and the first layer, 8 adds + 8 FMAs for the odd half)
// instead of the 56 of the composed 4 x 2 form.
template <int S>
struct Dft<8, S> {
    static __device__ __forceinline__ void run(cplx (&v)[8])
    {
        cplx a[4], b[4];
#pragma unroll
        for (int n = 0; n < 4; ++n) {
            a[n] = cadd(v[n], v[n + 4]);
            b[n] = csub(v[n], v[n + 4]);
        }
        dft8_tail<S>(a, b, v);
    }
};

template <int R>
struct Split {
    static constexpr int P = (R % 3 == 0) ? 3 : ((R % 4 == 0) ? 4 : 2);
};

// Composite radix R = P*Q (Cooley-Tukey, natural order in and out):
//   X[k1 + P*k2] = sum_{n2<Q} W_Q^{n2 k2} W_R^{n2 k1} sum_{n1<P} x[n2 + Q*n1] W_P^{n1 k1}
template <int R, int S>
struct Dft {
    static constexpr int P = Split<R>::P, Q = R / P;
    static __device__ __forceinline__ void run(cplx (&v)[R])
    {
        cplx t[Q][P];
        static_for<0, Q>([&](auto n2c) {
            constexpr int n2 = decltype(n2c)::value;
            cplx u[P];
#pragma unroll
            for (int n1 = 0; n1 < P; ++n1) u[n1] = v[n2 + Q * n1];
            Dft<P, S>::run(u);
            static_for<0, P>([&](auto k1c) {
                constexpr int k1 = decltype(k1c)::value;
                t[n2][k1] = mul_w<R, n2 * k1, S>(u[k1]);
            });
        });
        static_for<0, P>([&](auto k1c) {
            constexpr int k1 = decltype(k1c)::value;
            cplx u[Q];
#pragma unroll
            for (int n2 = 0; n2 < Q; ++n2) u[n2] = t[n2][k1];
            Dft<Q, S>::run(u);
#pragma unroll
            for (int k2 = 0; k2 < Q; ++k2) v[k1 + P * k2] = u[k2];
        });
    }
};

// DFT of size A = 3*A1 whose inputs n in [A1, 2*A1) are zero: lo = x[0..A1), hi = x[2*A1..3*A1).
// With n = a + A1*t, k = 3c + d:  X[3c+d] = sum_a W_A1^{ac} W_A^{ad} (lo[a] + W_3^{2d} hi[a]).
template <int A, int S>
__device__ __forceinline__ void dft_pruned_in(const cplx (&lo)[A / 3], const cplx (&hi)[A / 3], cplx (&out)[A])
{
    constexpr int A1 = A / 3;
    constexpr double h = S * kHalfSqrt3;
    cplx z0[A1], z1[A1], z2[A1];
    static_for<0, A1>([&](auto ac) {
        constexpr int a = decltype(ac)::value;
        cplx l = lo[a], c = hi[a];
        cplx m = cmake(fma(-0.5, c.x, l.x), fma(-0.5, c.y, l.y));
        z0[a] = cadd(l, c);
        z1[a] = mul_w<A, a, S>(cmake(fma(h, c.y, m.x), fma(-h, c.x, m.y)));      // l + W3^2 c
        z2[a] = mul_w<A, 2 * a, S>(cmake(fma(-h, c.y, m.x), fma(h, c.x, m.y)));  // l + W3   c
    });
    Dft<A1, S>::run(z0);
    Dft<A1, S>::run(z1);
    Dft<A1, S>::run(z2);
#pragma unroll
    for (int c = 0; c < A1; ++c) {
        out[3 * c] = z0[c];
        out[3 * c + 1] = z1[c];
        out[3 * c + 2] = z2[c];
    }
}

// DFT of size A = 3*A1 of which only the outputs k in [0,A1) (lo) and [2*A1,3*A1) (hi) are formed.
// With n = 3a + d, k = c + A1*t:  X[c + A1 t] = sum_d W_3^{dt} W_A^{dc} sum_a in[3a+d] W_A1^{ac}.
template <int A, int S>
__device__ __forceinline__ void dft_pruned_out(const cplx (&in)[A], cplx (&lo)[A / 3], cplx (&hi)[A / 3])
{
    constexpr int A1 = A / 3;
    constexpr double h = S * kHalfSqrt3;
    cplx v0[A1], v1[A1], v2[A1];
#pragma unroll
    for (int a = 0; a < A1; ++a) {
        v0[a] = in[3 * a];
        v1[a] = in[3 * a + 1];
        v2[a] = in[3 * a + 2];
    }
    Dft<A1, S>::run(v0);
    Dft<A1, S>::run(v1);
    Dft<A1, S>::run(v2);
    static_for<0, A1>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        cplx p = v0[c], q = mul_w<A, c, S>(v1[c]), r = mul_w<A, 2 * c, S>(v2[c]);
        cplx t = cadd(q, r), u = csub(r, q);
        lo[c] = cadd(p, t);
        cplx m = cmake(fma(-0.5, t.x, p.x), fma(-0.5, t.y, p.y));
        hi[c] = cmake(fma(-h, u.y, m.x), fma(h, u.x, m.y));  // m + S*i*h*(r - q)
    });
}

// Radix-8 DFT of TWIDDLED inputs, X[k] = sum_n (w[n] v[n]) W_8^{S n k} with w[0] = 1, natural order in place.
// Decimation in frequency with the twiddle products fused into the first layer: for the pair (n, n+4)
//     a = w[n] v[n],   s = a + w[n+4] v[n+4]  (4 FMA),   d = a - w[n+4] v[n+4] = 2 a - s  (2 FMA)
// i.e. 6 FP64 instructions instead of 8 for the second product and the butterfly; with dft8_tail, 68 per transform
// against 84 for seven complex products followed by the composed 4 x 2 radix 8.
template <int S>
__device__ __forceinline__ void dft8_twiddled(cplx (&v)[8], const cplx (&w)[8])
{
    cplx a[4], b[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) {
        const cplx x = (n == 0) ? v[0] : cmul(v[n], w[n].x, w[n].y);
        const cplx y = v[n + 4], t = w[n + 4];
        a[n] = cmake(fma(-y.y, t.y, fma(y.x, t.x, x.x)), fma(y.y, t.x, fma(y.x, t.y, x.y)));  // x + t y
        b[n] = cmake(fma(2.0, x.x, -a[n].x), fma(2.0, x.y, -a[n].y));                          // x - t y
    }
    dft8_tail<S>(a, b, v);
}

}  // namespace gnl
