// gene_nl.cu -- C ABI (include/gene_nl.h): plan, batching, launch sequence, host streaming driver.
//
// One gene_nl_compute walks the phase space in CHUNKS = (w,s) slab x z-range x all v, and inside a
// chunk in BATCHES of v whose scratch (Z, P, Rchi; see nl_kernels.cuh) fits the plan's scratch budget
// (default 768 MiB per set -- far beyond the 126 MB L2 on purpose: measured on B200, long launches beat
// L2-sized batches; gene_nl_set_scratch_bytes changes it).  With chi_has_v = 0 the real-space chi
// fields of a chunk are formed once and reused by every v (SURVEY.md 7 "chi reuse").  The host entry
// points stream (w,s) slabs over several CUDA streams.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/gene_nl_bench.h"
#include "nl_fused.cuh"
#include "nl_fused2.cuh"
#include "nl_cluster.cuh"
#include "nl_group.cuh"
#include "nl_wa.cuh"
#include "nl_kernels.cuh"
#include "nl_pipe.cuh"

using gnl::cplx;

namespace {

thread_local std::string g_err;

void set_err(const std::string& s) { g_err = s; }

bool cuda_ok(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return true;
    set_err(std::string(what) + ": " + cudaGetErrorString(e));
    return false;
}

// ---- per-length kernel tables --------------------------------------------------------------------
struct XGeom { const cplx* src; cplx* Z; int nky0, nzb; long long vstride; double kxmin, kymin; };

typedef void (*xinv_fn)(const cplx*, cplx*, const cplx*, int, int, long long, double, double);
typedef void (*xfwd_fn)(const cplx*, cplx*, const cplx*, int, int, long long, double);
typedef void (*yreal_fn)(const cplx*, cplx*, const cplx*, int);
typedef void (*ybr_fn)(const cplx*, const cplx*, cplx*, const cplx*, int, int, int, int, const cplx*, const double*);
typedef void (*fused_fn)(const cplx*, cplx*, const cplx*, const cplx*, const cplx*, int, int, int, int, double, double,
                         double);

typedef void (*fused2_fn)(const cplx*, cplx*, const cplx*, const cplx*, int, int, int, int, double, double, double);
typedef void (*cluster_fn)(const cplx*, cplx*, const cplx*, const cplx*, const cplx*, int, int, int, double, double, double);

typedef void (*group_fn)(const cplx*, cplx*, const cplx*, const cplx*, const cplx*, const cplx*, cplx*, unsigned*, int, int, int,
                         double, double, double, const cplx*, const double*, int, int);

struct FusedKernel {
    fused_fn fn = nullptr;
    fused2_fn fn2 = nullptr;  // second-generation kernel (nl_fused2.cuh); used when available
    cluster_fn fnc = nullptr; // the plane spread over a thread-block cluster (nl_cluster.cuh); chi shared over v only
    group_fn fng = nullptr;   // the plane spread over a group of co-resident CTAs, hand-overs through L2 (nl_group.cuh)
    bool chiv = false;        // group kernel: chi per plane goes through the kernel too (no chi-side launches)
    bool wa = false;          // fng is the warp-autonomous form (nl_wa.cuh)
    int group = 1;            // CTAs per group
    size_t group_scratch = 0; // bytes of Z + P scratch per group
    int cluster = 1;          // CTAs per cluster
    size_t smem = 0;
    int nt = 0;
};

template <int AX, int BX, int AY, int NW>
FusedKernel make_cluster()
{
    using K = gnl::Clustered<AX, BX, AY, NW>;
    FusedKernel k;
    k.fnc = gnl::k_plane_cluster<AX, BX, AY, NW>;
    k.cluster = K::C;
    k.smem = K::SMEM_BYTES;
    k.nt = K::NT;
    return k;
}

template <int AX, int BX, int AY, int G, int NW, int NH, bool CHIV, bool EM = false, int BY = 8, int NPW = 3, int AX2 = 0, int BX2 = 0,
          int CK = 8>
FusedKernel make_group()
{
    using K = gnl::Grouped<AX, BX, AY, G, NW, NH, CHIV, BY, NPW, AX2, BX2, CK>;
    FusedKernel k;
    k.fng = gnl::k_plane_group<AX, BX, AY, G, NW, NH, CHIV, EM, BY, NPW, AX2, BX2, CK>;
    k.chiv = CHIV;
    k.group = G;
    k.group_scratch = sizeof(cplx) * K::GROUP_SCRATCH_CPLX;
    k.smem = K::SMEM_BYTES;
    k.nt = K::NT;
    return k;
}

template <int AX, int BX, int AY, int BY, int G, int NW, bool CHIV, bool EM, int NPW, bool PF, int AX2 = 0, int BX2 = 0>
FusedKernel make_wa()
{
    using K = gnl::WarpAuto<AX, BX, AY, BY, G, NW, CHIV, NPW, AX2, BX2>;
    FusedKernel k;
    k.fng = gnl::k_plane_wa<AX, BX, AY, BY, G, NW, CHIV, EM, NPW, PF, AX2, BX2>;
    k.wa = true;
    k.chiv = CHIV;
    k.group = G;
    k.group_scratch = sizeof(cplx) * K::GROUP_SCRATCH_CPLX;
    k.smem = K::SMEM_BYTES;
    k.nt = K::NT;
    return k;
}

// The warp-autonomous form of the group kernel (nl_wa.cuh): same groups and scratch, no CTA-wide barrier in the plane loop
bool find_wa(int nx, int ny, bool chi_has_v, bool em, FusedKernel* out)
{
    if (em) return false;   // (the composition of chi on the device stays with the group kernel)
    if (nx == 384 && ny == 192 && !chi_has_v) { *out = make_wa<24, 16, 24, 8, 4, 8, false, false, 3, true>(); return out->smem <= 227 * 1024; }
    if (nx == 768 && ny == 384 && !chi_has_v) { *out = make_wa<24, 32, 24, 16, 8, 8, false, false, 2, false>(); return out->smem <= 227 * 1024; }
    if (nx == 144 && ny == 144 && chi_has_v) { *out = make_wa<12, 12, 18, 8, 1, 8, true, false, 3, true>(); return out->smem <= 227 * 1024; }
    if (nx == 144 && ny == 144 && !chi_has_v) { *out = make_wa<12, 12, 18, 8, 1, 8, false, false, 3, true>(); return out->smem <= 227 * 1024; }
    return false;
}

// Planes beyond one SM: groups of G co-resident CTAs per plane, Z and P through L2
bool find_group(int nx, int ny, bool chi_has_v, bool em, FusedKernel* out)
{
    if (em) {  // chi composed on the device from phi_bar and A_par_bar
        if (nx == 384 && ny == 192) { *out = make_group<24, 16, 24, 4, 8, 2, false, true>(); return out->smem <= 227 * 1024; }
        if (nx == 144 && ny == 144) { *out = make_group<12, 12, 18, 1, 8, 1, false, true>(); return out->smem <= 227 * 1024; }
        return false;
    }
    if (nx == 384 && ny == 192 && !chi_has_v) { *out = make_group<24, 16, 24, 4, 8, 2, false>(); return out->smem <= 227 * 1024; }
    if (nx == 768 && ny == 384 && !chi_has_v) { *out = make_group<48, 16, 24, 8, 8, 4, false, false, 16, 2, 24, 32>(); return out->smem <= 227 * 1024; }
    if (nx == 144 && ny == 144 && chi_has_v) { *out = make_group<12, 12, 18, 1, 8, 1, true>(); return out->smem <= 227 * 1024; }
    if (nx == 144 && ny == 144 && !chi_has_v) { *out = make_group<12, 12, 18, 1, 8, 1, false>(); return out->smem <= 227 * 1024; }
    return false;
}

// Planes whose Z exceeds one SM but fits the shared memory of a portable cluster (8 CTAs): 384 x 192 (configs[2])
bool find_cluster(int nx, int ny, FusedKernel* out)
{
    if (nx == 384 && ny == 192) { *out = make_cluster<24, 16, 24, 8>(); return out->smem <= 227 * 1024; }
    return false;
}

template <int AX, int AY, int NW>
FusedKernel make_fused2()
{
    FusedKernel k;
    k.fn2 = gnl::k_plane_fused2<AX, AY, NW>;
    k.smem = gnl::Fused2<AX, AY, NW>::SMEM_BYTES;
    k.nt = NW * 32;
    return k;
}

// nky0 a multiple of 32 (Ny = 96) and Nx = 8 AX <= 192: the warp-uniform-twiddle kernel
bool find_fused2(int nx, int ny, FusedKernel* out)
{
    if (ny != 96) return false;
    switch (nx) {
    case 48: *out = make_fused2<6, 12, 8>(); break;
    case 96: *out = make_fused2<12, 12, 8>(); break;
    case 192: *out = make_fused2<24, 12, 8>(); break;
    default: return false;
    }
    return out->smem <= 227 * 1024;
}

template <int AX, int AY, int NW>
FusedKernel make_fused()
{
    FusedKernel k;
    k.fn = gnl::k_plane_fused<AX, AY, NW>;
    k.smem = gnl::Fused<AX, AY, NW>::SMEM_BYTES;
    k.nt = NW * 32;
    return k;
}

// Planes whose half-transformed form fits in shared memory (Nx = 8 AX <= 192, Ny = 8 AY <= 96).
bool find_fused(int nx, int ny, FusedKernel* out)
{
    const int key = nx * 1000 + ny;
    switch (key) {
#define GNL_FUSED_CASE(AX, AY) case (8 * AX) * 1000 + 8 * AY: *out = make_fused<AX, AY, 8>(); break;
        GNL_FUSED_CASE(3, 3) GNL_FUSED_CASE(3, 6) GNL_FUSED_CASE(3, 12)
        GNL_FUSED_CASE(6, 3) GNL_FUSED_CASE(6, 6) GNL_FUSED_CASE(6, 12)
        GNL_FUSED_CASE(12, 3) GNL_FUSED_CASE(12, 6) GNL_FUSED_CASE(12, 12)
        GNL_FUSED_CASE(24, 3) GNL_FUSED_CASE(24, 6) GNL_FUSED_CASE(24, 12)
#undef GNL_FUSED_CASE
    default: return false;
    }
    return out->smem <= 227 * 1024;
}

typedef void (*xinvp_fn)(const cplx*, cplx*, const cplx*, int, int, long long, double, double, int);
struct XKernels {
    int nx, ck, nt;
    int ck_inv = 0, nt_inv = 0;  // k_xinv's own tile width / threads when they differ from k_xfwd's (0: the same)
    size_t smem_inv, smem_fwd;
    xinv_fn inv;
    xfwd_fn fwd;
    xinvp_fn invp_zt = nullptr;  // the same, storing Z transposed (for k_ybracket_t); may use fewer columns per tile
    int ck_zt = 0;
    size_t smem_invp_zt = 0;
    xinvp_fn invp = nullptr;  // pipelined persistent version (nl_pipe.cuh)
    size_t smem_invp = 0;
    int cap_invp = 0;         // its grid (resident CTAs); 0: use the first-generation kernel
};
typedef void (*ybrcv_fn)(const cplx*, const cplx*, cplx*, const cplx*, int);
typedef void (*ybrt_fn)(const cplx*, const cplx*, cplx*, const cplx*, int, int, int);
struct YKernels {
    int ny, rp, rt, nt;
    size_t smem_br, smem_real;
    ybr_fn br;
    ybr_fn br_em;  // chi = phi_bar - v_par A_par_bar composed in the bracket
    ybrt_fn br_t = nullptr;  // g side read from the transposed Z (tiles of 8 row pairs, 128 threads)
    size_t smem_t = 0;
    int rp_t = 8, nt_t = 128;
    ybrcv_fn br_cv;  // chi per plane: its y-synthesis fused into the bracket kernel (no R round trip)
    size_t smem_cv;
    int rp_cv;
    yreal_fn real;
};

template <int NX, int A, int B, int CK, int NT>
XKernels make_x()
{
    XKernels k;
    k.nx = NX; k.ck = CK; k.nt = NT;
    k.smem_inv = sizeof(cplx) * (size_t)(A * gnl::Tile<A, B>::BP + 2 * CK * gnl::Tile<A, B>::STRIDE);
    k.smem_fwd = sizeof(cplx) * (size_t)(A * gnl::Tile<A, B>::BP + CK * gnl::Tile<A, B>::STRIDE);
    k.inv = gnl::k_xinv<NX, A, B, CK, NT>;
    k.fwd = gnl::k_xfwd<NX, A, B, CK, NT>;
    k.invp = gnl::k_xinv_p<NX, A, B, CK, NT, false>;
    constexpr int CKZ = (NX >= 768) ? 2 : CK;  // transposed stores are 128 B runs for any CK: small tiles where smem is tight
    k.invp_zt = gnl::k_xinv_p<NX, A, B, CKZ, NT, true>;
    k.ck_zt = CKZ;
    k.smem_invp_zt = gnl::XInvP<NX, A, B, CKZ, NT>::SMEM_BYTES;
    k.smem_invp = gnl::XInvP<NX, A, B, CK, NT>::SMEM_BYTES;
    return k;
}
template <int NY, int A, int B, int RP, int NT>
YKernels make_y()
{
    YKernels k;
    k.ny = NY; k.rp = RP; k.rt = 2 * RP; k.nt = NT;
    k.smem_br = sizeof(cplx) * (size_t)(2 * RP * gnl::Tile<A, B>::FLAT);  // exchange tiles only (twiddles come through L1)
    k.smem_real = k.smem_br;
    k.br = gnl::k_ybracket<NY, A, B, RP, NT, false>;
    k.br_em = gnl::k_ybracket<NY, A, B, RP, NT, true>;
    constexpr int RPT = (NY >= 384) ? 4 : 8, NTT = (NY >= 384) ? 64 : 128;
    k.br_t = gnl::k_ybracket_t<NY, A, B, NTT, RPT>;
    k.smem_t = gnl::YBracketT<NY, A, B, NTT, RPT>::SMEM_BYTES;
    k.rp_t = RPT; k.nt_t = NTT;
    constexpr int RPC = (RP >= 8) ? RP / 2 : RP;  // twice the exchange tiles per pair: fewer pairs per CTA
    k.br_cv = gnl::k_ybracket_cv<NY, A, B, RPC, NT>;
    k.smem_cv = sizeof(cplx) * (size_t)(4 * RPC * gnl::Tile<A, B>::FLAT);
    k.rp_cv = RPC;
    k.real = gnl::k_yreal<NY, A, B, 2 * RP, NT>;
    return k;
}

bool find_x(int nx, XKernels* out)
{
    switch (nx) {
    case 24: *out = make_x<24, 3, 8, 8, 128>(); return true;
    case 48: *out = make_x<48, 6, 8, 8, 128>(); return true;
    case 96: *out = make_x<96, 12, 8, 8, 128>(); return true;
    case 144: *out = make_x<144, 12, 12, 8, 128>(); return true;
    case 192: *out = make_x<192, 24, 8, 8, 128>(); return true;
    case 288: *out = make_x<288, 18, 16, 4, 128>(); return true;
    case 384: *out = make_x<384, 24, 16, 4, 128>(); return true;
    case 576: *out = make_x<576, 24, 24, 4, 128>(); return true;
    case 1152: *out = make_x<1152, 36, 32, 4, 128>(); return true;
    case 1536: *out = make_x<1536, 48, 32, 2, 128>(); return true;
    case 768: *out = make_x<768, 24, 32, 4, 128>();
        // row-major Z in 128 B pieces: 8 columns per CTA, the two signs one after the other through the same 8 tiles
        // of E (measured on B200, configs[3]: k_xinv 36.0 -> 32.7 ms)
        out->inv = gnl::k_xinv<768, 24, 32, 8, 128, true>;
        out->ck_inv = 8; out->nt_inv = 128;
        return true;
    default: return false;
    }
}
// Row pairs per CTA must divide Nx/2; Nx/2 is a multiple of 12 for every supported Nx.
bool find_y(int ny, int nx, YKernels* out)
{
    const bool rp8 = (nx / 2) % 8 == 0;  // 8 row pairs per CTA when they divide Nx/2, else 4
    switch (ny) {
    case 24: *out = rp8 ? make_y<24, 3, 8, 8, 64>() : make_y<24, 3, 8, 4, 64>(); return true;
    case 48: *out = rp8 ? make_y<48, 6, 8, 8, 64>() : make_y<48, 6, 8, 4, 64>(); return true;
    case 96: *out = rp8 ? make_y<96, 12, 8, 8, 64>() : make_y<96, 12, 8, 4, 64>(); return true;
    case 144: *out = rp8 ? make_y<144, 12, 12, 8, 96>() : make_y<144, 12, 12, 4, 96>(); return true;
    case 192: *out = make_y<192, 12, 16, 4, 64>(); return true;
    case 288: *out = make_y<288, 18, 16, 4, 64>(); return true;
    case 384: *out = make_y<384, 24, 16, 4, 64>(); return true;
    case 576: *out = make_y<576, 24, 24, 4, 96>(); return true;
    default: return false;
    }
}

struct Scratch {
    cplx *Z = nullptr, *P = nullptr, *R = nullptr;
    cplx* GS = nullptr;       // group kernel: Z + P of every group's current plane (L2 resident)
    unsigned* cnt = nullptr;  // group kernel: two hand-over counters per group
    size_t r2off = 0;         // em on a plane kernel: where A_par_bar's real-space fields start in R (in values)
};

// Optional per-launch CUDA-event timing (gene_nl_compute_profiled): kernel classes
enum { K_XINV = 0, K_YREAL = 1, K_YBRACKET = 2, K_XFWD = 3, K_FUSED = 4, K_CLASSES = 5 };
struct Profiler {
    cudaStream_t st;
    std::vector<cudaEvent_t> ev;  // pairs (before, after)
    std::vector<int> cls;
    cudaEvent_t begin(int c)
    {
        cudaEvent_t a, b;
        cudaEventCreate(&a);
        cudaEventCreate(&b);
        ev.push_back(a);
        ev.push_back(b);
        cls.push_back(c);
        cudaEventRecord(a, st);
        return b;
    }
};
#define GNL_LAUNCH(prof, c, call)                          \
    do {                                                    \
        cudaEvent_t e_ = (prof) ? (prof)->begin(c) : nullptr; \
        call;                                               \
        if (prof) cudaEventRecord(e_, (prof)->st);          \
    } while (0)

struct HostStage {  // per-stream staging of one chunk for gene_nl_compute_host
    cudaStream_t stream = nullptr;
    cplx *g = nullptr, *rhs = nullptr, *chi = nullptr, *apar = nullptr;
    Scratch scr;
};

}  // namespace

struct gene_nl_plan {
    int nx0, nky0, nz, nv, nw, nspec, chi_has_v;
    bool zt = false;          // g side through the transposed Z: k_xinv_p<ZT> + k_ybracket_t (chi shared over v only)
    int cap_invp_zt = 0;
    bool fuse_chi_y = false;  // chi_has_v = 1 on the batched path: chi's y-synthesis inside k_ybracket_cv
    bool em = false;          // created with chi_has_v = 2: phi_bar and A_par_bar are supplied, chi is composed on device
    double* vp_dev = nullptr; // em: v_par coefficients, nv * nspec
    double kxmin, kymin;
    int Nx, Ny;
    size_t M;       // modes per plane
    long long planes;
    int nzb, nvb;   // chunk z-extent and batch v-extent
    XKernels xk;
    YKernels yk;
    FusedKernel fk;
    FusedKernel gk;           // the group kernel for this plane size, if there is one
    int gk_grid = 0;          // its grid: co-resident groups x CTAs per group
    FusedKernel wk;           // the warp-autonomous group kernel for this plane size, if there is one
    int wk_grid = 0;
    FusedKernel ck;           // the cluster kernel for this plane size, if there is one (gene_nl_set_plane_kernel)
    int ck_grid = 0;          // its grid: resident clusters x CTAs per cluster
    FusedKernel fk_auto;      // what gene_nl_create selected
    bool fused_auto = false;
    int fused_grid_auto = 0;
    bool fused = false;
    int fused_grid = 0;
    int nss = 1;      // fused: (w,s) slabs per launch (Rchi of that many slabs is kept)
    long long nbz = 1;  // fused: chi planes per k_xinv/k_yreal batch
    cplx *twx = nullptr, *twy = nullptr;
    Scratch scr;
    size_t zbytes, pbytes, rbytes;  // per scratch set
    size_t table_bytes;
    std::vector<HostStage> stages;  // lazily created by gene_nl_compute_host
    int device;
    size_t budget = (size_t)768 << 20;  // scratch budget per set (gene_nl_set_scratch_bytes)
    bool budget_set = false;            // explicit budget: it also bounds the fused path's chi cache
    double* vp_pinned = nullptr;        // em: host staging of v_par (pinned), guarded by vp_event
    cudaEvent_t vp_event = nullptr;
};

namespace {

bool alloc_scratch(size_t zbytes, size_t pbytes, size_t rbytes, Scratch* s)
{
    if (!cuda_ok(cudaMalloc(&s->Z, zbytes), "cudaMalloc(Z)")) return false;
    if (!cuda_ok(cudaMalloc(&s->P, pbytes), "cudaMalloc(P)")) return false;
    if (!cuda_ok(cudaMalloc(&s->R, rbytes), "cudaMalloc(Rchi)")) return false;
    s->r2off = rbytes / (2 * sizeof(cplx));   // em: phi_bar's fields fill the first half, A_par_bar's the second
    return true;
}
bool alloc_scratch(gene_nl_plan* h, Scratch* s);
void free_scratch(Scratch* s)
{
    cudaFree(s->Z); cudaFree(s->P); cudaFree(s->R); cudaFree(s->GS); cudaFree(s->cnt);
    s->Z = s->P = s->R = s->GS = nullptr;
    s->cnt = nullptr;
}

bool upload_twiddles(int n, cplx** out)
{
    std::vector<cplx> t(n);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int k = 0; k < n; ++k) {
        long double ang = two_pi * (long double)k / (long double)n;
        t[k].x = (double)cosl(ang);
        t[k].y = (double)sinl(ang);
    }
    if (!cuda_ok(cudaMalloc(out, sizeof(cplx) * n), "cudaMalloc(twiddles)")) return false;
    return cuda_ok(cudaMemcpy(*out, t.data(), sizeof(cplx) * n, cudaMemcpyHostToDevice), "cudaMemcpy(twiddles)");
}

// W_N^j of every supported length into the __constant__ table read by the warp-uniform x stages
bool upload_const_twiddles()
{
    static const int lens[] = {24, 48, 96, 144, 192, 384, 768};
    std::vector<cplx> t(gnl::kCTwTotal);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int n : lens) {
        const int off = gnl::ctw_offset(n);
        for (int k = 0; k < n; ++k) {
            long double ang = two_pi * (long double)k / (long double)n;
            t[off + k].x = (double)cosl(ang);
            t[off + k].y = (double)sinl(ang);
        }
    }
    return cuda_ok(cudaMemcpyToSymbol(gnl::c_tw, t.data(), sizeof(cplx) * t.size()), "cudaMemcpyToSymbol(twiddles)");
}

// Batching for the plan's scratch budget.  Batched path: chunk = nzb z-planes x all v; batch = nzb x nvb planes whose
// scratch set fits the budget.  Fused path: nss (w,s) slabs per launch (their real-space chi is kept), nbz chi planes
// per k_xinv / k_yreal batch.  Sets nzb, nvb, nss, nbz and the byte sizes of one scratch set.
bool alloc_group_scratch(gene_nl_plan* h, Scratch* s)
{
    if (!h->fused || !h->fk.fng) return true;
    const int ngroup = h->fused_grid / h->fk.group;
    return cuda_ok(cudaMalloc(&s->GS, h->fk.group_scratch * (size_t)ngroup), "cudaMalloc(group scratch)") &&
           cuda_ok(cudaMalloc(&s->cnt, sizeof(unsigned) * 2 * (size_t)ngroup), "cudaMalloc(group counters)");
}
bool alloc_scratch(gene_nl_plan* h, Scratch* s)
{
    return alloc_scratch(h->zbytes, h->pbytes, h->rbytes, s) && alloc_group_scratch(h, s);
}

void configure_batching(gene_nl_plan* h)
{
    const int nz = h->nz, nv = h->nv;
    const size_t W2 = 2 * (size_t)h->nky0;
    const size_t zpp = sizeof(cplx) * h->Nx * W2, ppp = zpp / 2, rpp = sizeof(cplx) * (size_t)h->Nx * h->Ny;
    const size_t budget = h->budget;
    if (h->fused && h->fk.chiv) {   // chi per plane inside the plane kernel: no chi-side scratch, all slabs in one launch
        size_t nss = (size_t)h->nw * h->nspec;
        while (nss > 1 && nss * (size_t)nz * nv >= ((size_t)1 << 31)) nss /= 2;   // 32-bit plane counters in the kernels
        if (h->budget_set) {   // an explicit budget still bounds the planes per launch (ragged launches in tests)
            const size_t per_slab = (size_t)nz * nv * (zpp + ppp);
            size_t cap = budget / per_slab;
            if (cap < 1) cap = 1;
            if (nss > cap) nss = cap;
        }
        h->nss = (int)nss;
        h->nbz = 1;
        h->nzb = nz; h->nvb = nv;
        h->zbytes = h->pbytes = h->rbytes = 256;
        return;
    }
    if (h->fused) {
        const size_t cps = (size_t)nz * (h->chi_has_v ? nv : 1);          // chi planes per slab
        const size_t rcap = h->budget_set ? budget : (size_t)2 << 30;     // real-space chi kept per launch
        size_t nss = rcap / (cps * rpp * (h->em ? 2 : 1));
        if (nss < 1) nss = 1;
        if (nss > (size_t)h->nw * h->nspec) nss = (size_t)h->nw * h->nspec;
        while (nss > 1 && nss * (size_t)nz * nv >= ((size_t)1 << 31)) nss /= 2;   // 32-bit plane counters in the kernels
        h->nss = (int)nss;
        const size_t zcap = (h->budget_set && budget < ((size_t)64 << 20)) ? budget : (size_t)64 << 20;
        size_t nbz = zcap / zpp;
        if (nbz < 1) nbz = 1;
        if (nbz > cps * nss) nbz = cps * nss;
        h->nbz = (long long)nbz;
        h->nzb = nz; h->nvb = nv;
        h->zbytes = zpp * nbz;
        h->pbytes = 256;
        h->rbytes = rpp * cps * nss * (h->em ? 2 : 1);   // em: phi_bar's fields, then A_par_bar's
        return;
    }
    int nzb = nz;
    if (!h->chi_has_v) {
        while (nzb > 1 && (size_t)nzb * rpp * (h->em ? 2 : 1) > budget / 4) nzb = (nzb + 1) / 2;
    }
    const size_t per_plane = zpp + ppp + (h->chi_has_v ? rpp : 0);
    while (nzb > 1 && (size_t)nzb * per_plane > budget / 2) nzb = (nzb + 1) / 2;
    const size_t fixed = h->chi_has_v ? 0 : (size_t)nzb * rpp * (h->em ? 2 : 1);
    long long nvb = (long long)((budget > fixed ? budget - fixed : 0) / ((size_t)nzb * per_plane));
    if (nvb < 1) nvb = 1;
    if (nvb > nv) nvb = nv;
    h->nzb = nzb; h->nvb = (int)nvb;
    const size_t nb = (size_t)nzb * nvb;
    h->zbytes = zpp * nb;
    h->pbytes = ppp * nb;
    h->rbytes = rpp * (h->chi_has_v ? nb : (size_t)nzb * (h->em ? 2 : 1));
}

template <class K>
bool set_smem(K fn, size_t bytes, const char* name)
{
    if (bytes > 227 * 1024) {
        set_err(std::string(name) + ": shared memory request exceeds 227 KB");
        return false;
    }
    return cuda_ok(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes), name);
}

// k_xinv over `ntiles` tiles: the pipelined persistent kernel when enabled, else one CTA per tile
#define GNL_XINV(prof, st, ntiles, SRC, ZZ, NZB, VSTR)                                                                           \
    do {                                                                                                                        \
        if (h->xk.cap_invp > 0)                                                                                                 \
            GNL_LAUNCH(prof, K_XINV, (h->xk.invp<<<((ntiles) < h->xk.cap_invp ? (ntiles) : h->xk.cap_invp), h->xk.nt, h->xk.smem_invp, st>>>( \
                                         SRC, ZZ, h->twx, h->nky0, NZB, VSTR, h->kxmin, h->kymin, (ntiles))));                   \
        else                                                                                                                    \
            GNL_LAUNCH(prof, K_XINV, (h->xk.inv<<<(h->xk.ck_inv ? (ntiles) * h->xk.ck / h->xk.ck_inv : (ntiles)), h->xk.nt_inv ? h->xk.nt_inv : h->xk.nt, h->xk.smem_inv, st>>>(SRC, ZZ, h->twx, h->nky0, NZB, VSTR, h->kxmin, h->kymin))); \
    } while (0)

// Enqueue one chunk: planes (zi in [0,nzc), vi in [0,nv)), plane offset zi + vstride*vi from g/rhs;
// chi planes zi (+ cvstride*vi if chi_has_v) from chi.  Returns number of launches or -1.
int enqueue_chunk(gene_nl_plan* h, const Scratch& s, const cplx* chi, long long cvstride, const cplx* g,
                  cplx* rhs, long long vstride, int nzc, double scale, cudaStream_t st, Profiler* prof = nullptr,
                  const cplx* apar = nullptr, const double* vp = nullptr)
{
    const XKernels& xk = h->xk;
    const YKernels& yk = h->yk;
    const int xt = h->nky0 / xk.ck;            // column tiles per plane
    const int yt_pairs = (h->Nx / 2) / yk.rp;  // row-pair tiles per plane
    const int yt_rows = h->Nx / yk.rt;         // row tiles per plane (k_yreal)
    const double coef = scale / (2.0 * (double)h->Nx * (double)h->Ny);
    int launches = 0;
    // real-space chi of the chunk beyond a third of L2: walk the batch v-fastest (see k_ybracket)
    const int vfast = !h->chi_has_v && (size_t)nzc * h->Nx * h->Ny * sizeof(cplx) > ((size_t)40 << 20);
    if (!h->chi_has_v) {
        GNL_XINV(prof, st, nzc * xt, chi, s.Z, nzc, 0);
        GNL_LAUNCH(prof, K_YREAL, (yk.real<<<nzc * yt_rows, yk.nt, yk.smem_real, st>>>(s.Z, s.R, h->twy, h->Nx)));
        launches += 2;
    }
    cplx* R2 = nullptr;
    if (apar) {  // em: the same two kernels on A_par_bar; its real-space fields follow those of phi_bar in R
        R2 = s.R + (size_t)h->nzb * h->Nx * h->Ny;
        GNL_XINV(prof, st, nzc * xt, apar, s.Z, nzc, 0);
        GNL_LAUNCH(prof, K_YREAL, (yk.real<<<nzc * yt_rows, yk.nt, yk.smem_real, st>>>(s.Z, R2, h->twy, h->Nx)));
        launches += 2;
    }
    for (int v0 = 0; v0 < h->nv; v0 += h->nvb) {
        const int nvc = (h->nv - v0 < h->nvb) ? h->nv - v0 : h->nvb;
        const int nb = nzc * nvc;
        const size_t off = (size_t)v0 * (size_t)vstride * h->M;
        if (h->chi_has_v && h->fuse_chi_y) {
            // chi per plane: its x-synthesis goes to the R buffer (large enough: Nx*Ny >= Nx*2nky0 per plane) and its
            // y-synthesis runs inside k_ybracket_cv
            const size_t coff = (size_t)v0 * (size_t)cvstride * h->M;
            GNL_XINV(prof, st, nb * xt, chi + coff, s.R, nzc, cvstride);
            GNL_XINV(prof, st, nb * xt, g + off, s.Z, nzc, vstride);
            GNL_LAUNCH(prof, K_YBRACKET, (yk.br_cv<<<nb * ((h->Nx / 2) / yk.rp_cv), yk.nt, yk.smem_cv, st>>>(s.Z, s.R, s.P, h->twy, h->Nx)));
            GNL_LAUNCH(prof, K_XFWD, (xk.fwd<<<nb * xt, xk.nt, xk.smem_fwd, st>>>(s.P, rhs + off, h->twx, h->nky0, nzc, vstride, coef)));
            launches += 4;
            continue;
        }
        if (h->chi_has_v) {
            const size_t coff = (size_t)v0 * (size_t)cvstride * h->M;
            GNL_XINV(prof, st, nb * xt, chi + coff, s.Z, nzc, cvstride);
            GNL_LAUNCH(prof, K_YREAL, (yk.real<<<nb * yt_rows, yk.nt, yk.smem_real, st>>>(s.Z, s.R, h->twy, h->Nx)));
            launches += 2;
        }
        if (h->zt && !apar) {
            const int ntot = nb * (h->nky0 / xk.ck_zt);
            GNL_LAUNCH(prof, K_XINV, (xk.invp_zt<<<(ntot < h->cap_invp_zt ? ntot : h->cap_invp_zt), xk.nt, xk.smem_invp_zt, st>>>(g + off, s.Z, h->twx, h->nky0, nzc, vstride, h->kxmin, h->kymin, ntot)));
            GNL_LAUNCH(prof, K_YBRACKET, (yk.br_t<<<nb * ((h->Nx / 2) / yk.rp_t), yk.nt_t, yk.smem_t, st>>>(s.Z, s.R, s.P, h->twy, h->Nx, nzc, vfast)));
            GNL_LAUNCH(prof, K_XFWD, (xk.fwd<<<nb * xt, xk.nt, xk.smem_fwd, st>>>(s.P, rhs + off, h->twx, h->nky0, nzc, vstride, coef)));
            launches += 3;
            continue;
        }
        GNL_XINV(prof, st, nb * xt, g + off, s.Z, nzc, vstride);
        if (apar)
            GNL_LAUNCH(prof, K_YBRACKET, (yk.br_em<<<nb * yt_pairs, yk.nt, yk.smem_br, st>>>(s.Z, s.R, s.P, h->twy, h->Nx, nzc, 0, vfast, R2, vp + v0)));
        else
            GNL_LAUNCH(prof, K_YBRACKET, (yk.br<<<nb * yt_pairs, yk.nt, yk.smem_br, st>>>(s.Z, s.R, s.P, h->twy, h->Nx, nzc, h->chi_has_v, vfast, nullptr, nullptr)));
        GNL_LAUNCH(prof, K_XFWD, (xk.fwd<<<nb * xt, xk.nt, xk.smem_fwd, st>>>(s.P, rhs + off, h->twx, h->nky0, nzc, vstride, coef)));
        launches += 3;
    }
    if (!cuda_ok(cudaGetLastError(), "kernel launch")) return -1;
    return launches;
}

// Enqueue `nslab` contiguous (w,s) slabs (standard strides: v stride nz planes).  Returns launches or -1.
int enqueue_slabs(gene_nl_plan* h, const Scratch& s, const cplx* chi, const cplx* g, cplx* rhs, int nslab,
                  double scale, cudaStream_t st, Profiler* prof = nullptr, const cplx* apar = nullptr, int slab0 = 0)
{
    int launches = 0;
    if (h->fused) {
        const XKernels& xk = h->xk;
        const YKernels& yk = h->yk;
        const int xt = h->nky0 / xk.ck, yt_rows = h->Nx / yk.rt;
        const double coef = scale / (2.0 * (double)h->Nx * (double)h->Ny);
        for (int s0 = 0; s0 < nslab; s0 += h->nss) {
            const int ns = (nslab - s0 < h->nss) ? nslab - s0 : h->nss;
            const size_t cps = (size_t)h->nz * (h->chi_has_v ? h->nv : 1);  // chi planes per slab
            const size_t nchi = cps * ns;
            const cplx* chi0 = chi + (size_t)s0 * cps * h->M;
            for (size_t q0 = 0; q0 < nchi && !h->fk.chiv; q0 += (size_t)h->nbz) {   // chiv: chi goes through the plane kernel
                const int nb = (int)((nchi - q0 < (size_t)h->nbz) ? nchi - q0 : (size_t)h->nbz);
                GNL_XINV(prof, st, nb * xt, chi0 + q0 * h->M, s.Z, nb, 0);
                GNL_LAUNCH(prof, K_YREAL, (yk.real<<<nb * yt_rows, yk.nt, yk.smem_real, st>>>(s.Z, s.R + q0 * (size_t)h->Nx * h->Ny, h->twy, h->Nx)));
                launches += 2;
                if (apar) {  // em: the same two kernels on A_par_bar; its real-space fields fill the second half of R
                    cplx* R2 = s.R + s.r2off;
                    GNL_XINV(prof, st, nb * xt, apar + (size_t)s0 * cps * h->M + q0 * h->M, s.Z, nb, 0);
                    GNL_LAUNCH(prof, K_YREAL, (yk.real<<<nb * yt_rows, yk.nt, yk.smem_real, st>>>(s.Z, R2 + q0 * (size_t)h->Nx * h->Ny, h->twy, h->Nx)));
                    launches += 2;
                }
            }
            const size_t goff = (size_t)s0 * h->nz * h->nv * h->M;
            long long T = (long long)ns * h->nz * h->nv;
            int grid = (T < h->fused_grid) ? (int)T : h->fused_grid;
            if (h->fk.fng) {
                // cooperative launch (the CTAs of a group wait on one another); whole groups only
                const int G = h->fk.group;
                long long ngr = (T < h->fused_grid / G) ? T : h->fused_grid / G;
                cudaMemsetAsync(s.cnt, 0, sizeof(unsigned) * 2 * (size_t)(h->fused_grid / G), st);
                cudaLaunchConfig_t cfg = {};
                cudaLaunchAttribute at[1];
                cfg.gridDim = dim3((unsigned)(ngr * G));
                cfg.blockDim = dim3((unsigned)h->fk.nt);
                cfg.dynamicSmemBytes = h->fk.smem;
                cfg.stream = st;
                at[0].id = cudaLaunchAttributeCooperative;
                at[0].val.cooperative = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                // (a persisting-L2 access window over the scratch was measured on B200: the kernel gains 1.5 %, the
                // chi-side kernels lose more to the carve-out: not used)
                GNL_LAUNCH(prof, K_FUSED, (cudaLaunchKernelEx(&cfg, h->fk.fng, g + goff, (cplx*)(rhs + goff), (const cplx*)s.R, (const cplx*)(h->fk.chiv ? chi + goff : nullptr), (const cplx*)h->twx, (const cplx*)h->twy, s.GS, s.cnt, h->nz, h->nv, ns, h->kxmin, h->kymin, coef,
                                                              (const cplx*)(apar ? s.R + s.r2off : nullptr), (const double*)(apar ? h->vp_dev : nullptr), h->nw, slab0 + s0)));
            } else if (h->fk.fnc) {
                // whole clusters only; a cluster walks planes with the stride of the cluster count
                const int C = h->fk.cluster;
                long long ncl = (T < h->fused_grid / C) ? T : h->fused_grid / C;
                cudaLaunchConfig_t cfg = {};
                cudaLaunchAttribute at[1];
                cfg.gridDim = dim3((unsigned)(ncl * C));
                cfg.blockDim = dim3((unsigned)h->fk.nt);
                cfg.dynamicSmemBytes = h->fk.smem;
                cfg.stream = st;
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = (unsigned)C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                GNL_LAUNCH(prof, K_FUSED, (cudaLaunchKernelEx(&cfg, h->fk.fnc, g + goff, (cplx*)(rhs + goff), (const cplx*)s.R, (const cplx*)h->twx, (const cplx*)h->twy, h->nz, h->nv, ns, h->kxmin, h->kymin, coef)));
            } else if (h->fk.fn2)
                GNL_LAUNCH(prof, K_FUSED, (h->fk.fn2<<<grid, h->fk.nt, h->fk.smem, st>>>(g + goff, rhs + goff, s.R, h->twy, h->nz, h->nv, ns, h->chi_has_v, h->kxmin, h->kymin, coef)));
            else
                GNL_LAUNCH(prof, K_FUSED, (h->fk.fn<<<grid, h->fk.nt, h->fk.smem, st>>>(g + goff, rhs + goff, s.R, h->twx, h->twy, h->nz, h->nv, ns, h->chi_has_v, h->kxmin, h->kymin, coef)));
            launches += 1;
        }
        if (!cuda_ok(cudaGetLastError(), "kernel launch")) return -1;
        return launches;
    }
    for (int sl = 0; sl < nslab; ++sl) {
        const Scratch& sc = s;
        cudaStream_t str = st;
        for (int z0 = 0; z0 < h->nz; z0 += h->nzb) {
            const int nzc = (h->nz - z0 < h->nzb) ? h->nz - z0 : h->nzb;
            const size_t goff = ((size_t)z0 + (size_t)h->nz * h->nv * sl) * h->M;
            const size_t coff = h->chi_has_v ? goff : ((size_t)z0 + (size_t)h->nz * sl) * h->M;
            // em: slab sl = w + nw * species; its v_par coefficients are vp_dev[nv * species ..]
            int n = enqueue_chunk(h, sc, chi + coff, h->nz, g + goff, rhs + goff, h->nz, nzc, scale, str, prof,
                                  apar ? apar + coff : nullptr, apar ? h->vp_dev + (size_t)h->nv * ((slab0 + sl) / h->nw) : nullptr);
            if (n < 0) return -1;
            launches += n;
        }
    }
    return launches;
}

int chunks_per_slab(const gene_nl_plan* h) { return (h->nz + h->nzb - 1) / h->nzb; }

int launches_per_chunk(const gene_nl_plan* h)
{
    const int nbatch = (h->nv + h->nvb - 1) / h->nvb;
    return h->chi_has_v ? (h->fuse_chi_y ? 4 : 5) * nbatch : (h->em ? 4 : 2) + 3 * nbatch;
}

}  // namespace

extern "C" {

const char* gene_nl_last_error(void) { return g_err.c_str(); }

// internal (not in the header): lets the other translation units of the library set the same thread-local string
void gene_nl_set_error_(const char* msg) { g_err = msg ? msg : ""; }

gene_nl_plan* gene_nl_create(int nx0, int nky0, int nz, int nv, int nw, int nspec, double kxmin, double kymin,
                             int chi_has_v)
{
    g_err.clear();
    if (nx0 <= 0 || nky0 <= 0 || nz <= 0 || nv <= 0 || nw <= 0 || nspec <= 0 || (nx0 & 1) ||
        !std::isfinite(kxmin) || !std::isfinite(kymin)) {
        set_err("gene_nl_create: extents must be positive, nx0 even, kxmin/kymin finite");
        return nullptr;
    }
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice (no CUDA device: this library has no CPU fallback)")) return nullptr;
    gene_nl_plan* h = new gene_nl_plan();
    h->nx0 = nx0; h->nky0 = nky0; h->nz = nz; h->nv = nv; h->nw = nw; h->nspec = nspec;
    h->em = chi_has_v == GENE_NL_CHI_EM;
    h->chi_has_v = (chi_has_v && !h->em) ? 1 : 0;
    h->kxmin = kxmin; h->kymin = kymin;
    h->Nx = 3 * nx0 / 2; h->Ny = 3 * nky0;
    h->M = (size_t)nx0 * nky0;
    h->planes = (long long)nz * nv * nw * nspec;
    h->device = dev;
    if (!find_x(h->Nx, &h->xk) || !find_y(h->Ny, h->Nx, &h->yk)) {
        char buf[256];
        snprintf(buf, sizeof buf, "gene_nl_create: unsupported padded grid %dx%d (Nx in {24,48,96,144,192,288,384,576,768,1152,1536}, Ny in {24,48,96,144,192,288,384,576})", h->Nx, h->Ny);
        set_err(buf);
        delete h;
        return nullptr;
    }
    if (nky0 % h->xk.ck || (h->xk.ck_inv && nky0 % h->xk.ck_inv) || (h->Nx / 2) % h->yk.rp || h->Nx % h->yk.rt) {
        set_err("gene_nl_create: internal tiling does not divide the grid");
        delete h;
        return nullptr;
    }
    h->table_bytes = sizeof(cplx) * (size_t)(h->Nx + h->Ny);
    // the composition chi = phi_bar - v_par A_par_bar lives in k_ybracket (batched path)
    h->fused = !h->em && (find_fused2(h->Nx, h->Ny, &h->fk) || find_fused(h->Nx, h->Ny, &h->fk));
    // Planes beyond one SM.  The cluster kernel (nl_cluster.cuh) keeps Z and P out of HBM (1.03 x the algorithmic bytes,
    // ncu) but measured slower than the batched kernels on B200 (configs[2]: 8.2 ms against 7.2 ms: only 15 clusters of
    // 8 CTAs are co-resident on the 148 SMs, and the DSMEM hand-overs run at 18 B/clk/SM in series with the butterflies;
    // DESIGN.md sect. 6e), so it is selected on request only (gene_nl_set_plane_kernel).  The group kernel (nl_group.cuh)
    // replaced DSMEM by an L2-resident scratch and clusters by groups of a cooperative launch: see below.
    if (!h->fused && !h->em && !h->chi_has_v) find_cluster(h->Nx, h->Ny, &h->ck);
    if (!h->fused) find_group(h->Nx, h->Ny, h->chi_has_v != 0, h->em, &h->gk);
    if (!h->fused) find_wa(h->Nx, h->Ny, h->chi_has_v != 0, h->em, &h->wk);
    if (h->fused) {
        int sms = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        h->fused_grid = sms > 0 ? sms : 148;
    }
    configure_batching(h);

    bool ok = upload_twiddles(h->Nx, &h->twx) && upload_twiddles(h->Ny, &h->twy) && alloc_scratch(h, &h->scr) &&
              (!h->em || cuda_ok(cudaMalloc(&h->vp_dev, sizeof(double) * (size_t)nv * nspec), "cudaMalloc(v_par)")) &&
              (!h->em || set_smem(h->yk.br_em, h->yk.smem_br, "k_ybracket(em) smem")) &&
              set_smem(h->xk.inv, h->xk.smem_inv, "k_xinv smem") && set_smem(h->xk.fwd, h->xk.smem_fwd, "k_xfwd smem") &&
              set_smem(h->yk.br, h->yk.smem_br, "k_ybracket smem") && set_smem(h->yk.real, h->yk.smem_real, "k_yreal smem") &&
              (!h->ck.fnc || set_smem(h->ck.fnc, h->ck.smem, "k_plane_cluster smem")) &&
              (!h->gk.fng || set_smem(h->gk.fng, h->gk.smem, "k_plane_group smem")) &&
              (!h->wk.fng || set_smem(h->wk.fng, h->wk.smem, "k_plane_wa smem")) &&
              (!h->fused || (h->fk.fn2 ? set_smem(h->fk.fn2, h->fk.smem, "k_plane_fused2 smem")
                                       : set_smem(h->fk.fn, h->fk.smem, "k_plane_fused smem"))) &&
              upload_const_twiddles();
    if (ok && h->ck.fnc) {  // persistent clusters: as many as the device keeps resident at once
        int sms = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        cfg.gridDim = dim3((unsigned)(h->ck.cluster * ((sms > 0 ? sms : 148) / h->ck.cluster)));
        cfg.blockDim = dim3((unsigned)h->ck.nt);
        cfg.dynamicSmemBytes = h->ck.smem;
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)h->ck.cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int ncl = 0;
        if (cudaOccupancyMaxActiveClusters(&ncl, h->ck.fnc, &cfg) != cudaSuccess || ncl < 1) {
            cudaGetLastError();
            h->ck = FusedKernel();   // no cluster of that size fits this device: the option is not offered
        } else {
            h->ck_grid = ncl * h->ck.cluster;
        }
    }
    if (ok && h->gk.fng) {  // co-resident groups (cooperative launch)
        int sms = 0, occ = 0, coop = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->gk.fng, h->gk.nt, h->gk.smem) != cudaSuccess || occ < 1 ||
            sms < h->gk.group) {
            cudaGetLastError();
            h->gk = FusedKernel();
        } else {
            if (occ > 2) occ = 2;
            h->gk_grid = ((sms * occ) / h->gk.group) * h->gk.group;
        }
    }
    if (ok && h->wk.fng) {  // co-resident groups (cooperative launch), one CTA per SM
        int sms = 0, occ = 0, coop = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->wk.fng, h->wk.nt, h->wk.smem) != cudaSuccess || occ < 1 ||
            sms < h->wk.group) {
            cudaGetLastError();
            h->wk = FusedKernel();
        } else {
            h->wk_grid = (sms / h->wk.group) * h->wk.group;
        }
    }
    // The two optimisations of the batched path further down are decided for the batched path itself, i.e. for every
    // plane that does not fit one SM, whether or not a group kernel becomes the default next: enqueue_chunk consults them
    // only when the batched kernels run (gene_nl_set_plane_kernel(GENE_NL_KERNEL_BATCHED) on such a plan included).
    const bool one_sm = h->fused;
    if (ok && h->gk.fng && !h->fused) {
        // Planes beyond one SM with chi shared over v: the group kernel (Z and P through L2) is the default where it
        // exists.  Measured on B200 at configs[2]: 6.24 ms per step against 7.24 ms for the batched kernels and 8.18 ms
        // for the cluster kernel; DRAM traffic 1.07 x the algorithmic bytes (batched: about 4 x).
        free_scratch(&h->scr);
        h->fk = h->gk; h->fused = true; h->fused_grid = h->gk_grid;
        configure_batching(h);
        ok = alloc_scratch(h, &h->scr);
    }
    h->fk_auto = h->fk; h->fused_auto = h->fused; h->fused_grid_auto = h->fused_grid;
    if (ok && h->Nx <= 192) {
        // pipelined persistent x kernel; measured on B200: faster for Nx <= 192 (configs[4]: k_xinv 12.0 -> 10.2 ms),
        // equal at 384, slower at 768
        int sms = 0, occ = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (h->xk.smem_invp <= 227 * 1024 && set_smem(h->xk.invp, h->xk.smem_invp, "k_xinv_p smem") &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->xk.invp, h->xk.nt, h->xk.smem_invp) == cudaSuccess && occ > 0)
            h->xk.cap_invp = occ * sms;
    }
    if (ok && !h->chi_has_v && !h->em && !one_sm && (h->Nx / 2) % h->yk.rp_t == 0 && h->nky0 % h->xk.ck_zt == 0 &&
        h->Ny <= 192 && h->yk.smem_t <= 227 * 1024 && h->xk.smem_invp_zt <= 227 * 1024) {
        // measured on B200: 384 x 192 (configs[2]) 7.79 -> 7.19 ms; at Ny = 384 the 105 KB of exchange tiles of
        // k_ybracket_t cost more than the stores save (configs[3]: 101 -> 119 ms), so that size keeps the row-major Z
        int sms = 0, occ = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (set_smem(h->yk.br_t, h->yk.smem_t, "k_ybracket_t smem") &&
            set_smem(h->xk.invp_zt, h->xk.smem_invp_zt, "k_xinv_p<ZT> smem") &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->xk.invp_zt, h->xk.nt, h->xk.smem_invp_zt) == cudaSuccess && occ > 0) {
            h->zt = true;
            h->cap_invp_zt = occ * sms;
        }
    }
    if (ok && h->chi_has_v && !one_sm && (h->Nx / 2) % h->yk.rp_cv == 0 && h->yk.smem_cv <= 227 * 1024)
        h->fuse_chi_y = set_smem(h->yk.br_cv, h->yk.smem_cv, "k_ybracket_cv smem");
    if (!ok) {
        std::string keep = g_err;
        gene_nl_destroy(h);
        g_err = keep;
        return nullptr;
    }
    return h;
}

static void free_stages(gene_nl_plan* h)
{
    for (auto& s : h->stages) {
        cudaFree(s.g); cudaFree(s.rhs); cudaFree(s.chi); cudaFree(s.apar);
        free_scratch(&s.scr);
        if (s.stream) cudaStreamDestroy(s.stream);
    }
    h->stages.clear();
}

// The plan's tables, scratch and __constant__ twiddles live on the device it was created on
static bool on_plan_device(const gene_nl_plan* h)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) {
        set_err("the current CUDA device is not the one the plan was created on");
        return false;
    }
    return true;
}

void gene_nl_destroy(gene_nl_plan* h)
{
    if (!h) return;
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != h->device) cudaSetDevice(h->device);  // free on the owning device, then restore
    cudaDeviceSynchronize();
    free_stages(h);
    free_scratch(&h->scr);
    cudaFree(h->twx);
    cudaFree(h->twy);
    cudaFree(h->vp_dev);
    if (h->vp_pinned) cudaFreeHost(h->vp_pinned);
    if (h->vp_event) cudaEventDestroy(h->vp_event);
    if (cur >= 0 && cur != h->device) cudaSetDevice(cur);
    delete h;
}

int gene_nl_set_scratch_bytes(gene_nl_plan* h, size_t bytes)
{
    g_err.clear();
    if (!h) { set_err("NULL plan"); return GENE_NL_EINVAL; }
    if (bytes < ((size_t)1 << 20)) { set_err("gene_nl_set_scratch_bytes: the budget must be at least 1 MiB"); return GENE_NL_EINVAL; }
    if (!on_plan_device(h)) return GENE_NL_EINVAL;
    if (!cuda_ok(cudaDeviceSynchronize(), "cudaDeviceSynchronize")) return GENE_NL_ECUDA;
    const size_t old_budget = h->budget;
    const bool old_set = h->budget_set;
    free_stages(h);
    free_scratch(&h->scr);
    h->budget = bytes;
    h->budget_set = true;
    configure_batching(h);
    if (!alloc_scratch(h, &h->scr)) {  // fall back to the previous budget so that the plan stays usable
        std::string keep = g_err;
        free_scratch(&h->scr);
        h->budget = old_budget;
        h->budget_set = old_set;
        configure_batching(h);
        if (!alloc_scratch(h, &h->scr)) { free_scratch(&h->scr); }
        g_err = keep;
        return GENE_NL_ENOMEM;
    }
    return GENE_NL_OK;
}

int gene_nl_set_plane_kernel(gene_nl_plan* h, int kind)
{
    g_err.clear();
    if (!h) { set_err("NULL plan"); return GENE_NL_EINVAL; }
    if (kind != GENE_NL_KERNEL_AUTO && kind != GENE_NL_KERNEL_CLUSTER && kind != GENE_NL_KERNEL_GROUP && kind != GENE_NL_KERNEL_BATCHED &&
        kind != GENE_NL_KERNEL_WARP) {
        set_err("gene_nl_set_plane_kernel: unknown kind");
        return GENE_NL_EINVAL;
    }
    if (kind == GENE_NL_KERNEL_GROUP && !h->gk.fng) {
        set_err("gene_nl_set_plane_kernel: no group kernel for this plan (padded grids 384 x 192 [chi_has_v = 0 or EM], 768 x 384 [chi_has_v = 0], 144 x 144 [any chi]; a device with cooperative launch)");
        return GENE_NL_EUNSUPPORTED;
    }
    if (kind == GENE_NL_KERNEL_WARP && !h->wk.fng) {
        set_err("gene_nl_set_plane_kernel: no warp-autonomous group kernel for this plan (384 x 192 or 768 x 384 with chi shared over v, 144 x 144; not with GENE_NL_CHI_EM)");
        return GENE_NL_EUNSUPPORTED;
    }
    if (kind == GENE_NL_KERNEL_CLUSTER && !h->ck.fnc) {
        set_err("gene_nl_set_plane_kernel: no cluster kernel for this plan (384 x 192 padded grid, chi shared over v, a device that keeps clusters of 8 CTAs resident)");
        return GENE_NL_EUNSUPPORTED;
    }
    if (!on_plan_device(h)) return GENE_NL_EINVAL;
    if (!cuda_ok(cudaDeviceSynchronize(), "cudaDeviceSynchronize")) return GENE_NL_ECUDA;
    free_stages(h);
    free_scratch(&h->scr);
    if (kind == GENE_NL_KERNEL_CLUSTER) { h->fk = h->ck; h->fused = true; h->fused_grid = h->ck_grid; }
    else if (kind == GENE_NL_KERNEL_GROUP) { h->fk = h->gk; h->fused = true; h->fused_grid = h->gk_grid; }
    else if (kind == GENE_NL_KERNEL_WARP) { h->fk = h->wk; h->fused = true; h->fused_grid = h->wk_grid; }
    else if (kind == GENE_NL_KERNEL_BATCHED) { h->fk = FusedKernel(); h->fused = false; h->fused_grid = 0; }
    else { h->fk = h->fk_auto; h->fused = h->fused_auto; h->fused_grid = h->fused_grid_auto; }
    configure_batching(h);
    if (!alloc_scratch(h, &h->scr)) { free_scratch(&h->scr); return GENE_NL_ENOMEM; }
    return GENE_NL_OK;
}

static int check_ptrs(const void* chi, const void* g, void* rhs, size_t gbytes, size_t cbytes)
{
    if (!chi || !g || !rhs) { set_err("NULL array pointer"); return GENE_NL_EINVAL; }
    if (((uintptr_t)chi | (uintptr_t)g | (uintptr_t)rhs) & 15) { set_err("array pointers must be 16-byte aligned"); return GENE_NL_EINVAL; }
    const char *r0 = (const char*)rhs, *r1 = r0 + gbytes;
    const char *g0 = (const char*)g, *c0 = (const char*)chi;
    if ((g0 < r1 && r0 < g0 + gbytes) || (c0 < r1 && r0 < c0 + cbytes)) { set_err("rhs overlaps g or chi"); return GENE_NL_EINVAL; }
    return GENE_NL_OK;
}

static int compute_impl(gene_nl_plan* h, const void* chi_, const void* g_, void* rhs_, double scale, void* stream,
                        Profiler* prof)
{
    g_err.clear();
    if (!h) { set_err("NULL plan"); return GENE_NL_EINVAL; }
    if (h->em) { set_err("plan was created with GENE_NL_CHI_EM: call gene_nl_compute_em"); return GENE_NL_EINVAL; }
    if (!on_plan_device(h)) return GENE_NL_EINVAL;
    if (!h->scr.Z) { set_err("the plan has no scratch (an earlier gene_nl_set_scratch_bytes ran out of memory)"); return GENE_NL_ENOMEM; }
    const size_t gbytes = sizeof(cplx) * h->M * (size_t)h->planes;
    const size_t cbytes = h->chi_has_v ? gbytes : gbytes / h->nv;
    int rc = check_ptrs(chi_, g_, rhs_, gbytes, cbytes);
    if (rc) return rc;
    const cplx* chi = (const cplx*)chi_;
    const cplx* g = (const cplx*)g_;
    cplx* rhs = (cplx*)rhs_;
    cudaStream_t st = (cudaStream_t)stream;
    if (prof) prof->st = st;
    if (enqueue_slabs(h, h->scr, chi, g, rhs, h->nw * h->nspec, scale, st, prof) < 0) return GENE_NL_ECUDA;
    return GENE_NL_OK;
}

// em: v_par goes host -> plan-owned pinned staging -> device on `st`.  The staging buffer is reused by the next call,
// so this one waits (on the host) for the previous call's copy; the caller's array is free when the call returns.
static int stage_vpar(gene_nl_plan* h, const double* vpar_host, cudaStream_t st)
{
    const size_t n = (size_t)h->nv * h->nspec;
    if (!h->vp_pinned) {
        if (!cuda_ok(cudaMallocHost(&h->vp_pinned, sizeof(double) * n), "cudaMallocHost(v_par)")) return GENE_NL_ENOMEM;
        if (!cuda_ok(cudaEventCreateWithFlags(&h->vp_event, cudaEventDisableTiming), "cudaEventCreate")) return GENE_NL_ECUDA;
    } else if (!cuda_ok(cudaEventSynchronize(h->vp_event), "cudaEventSynchronize(v_par)")) {
        return GENE_NL_ECUDA;
    }
    std::memcpy(h->vp_pinned, vpar_host, sizeof(double) * n);
    if (!cuda_ok(cudaMemcpyAsync(h->vp_dev, h->vp_pinned, sizeof(double) * n, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync(v_par)") ||
        !cuda_ok(cudaEventRecord(h->vp_event, st), "cudaEventRecord(v_par)"))
        return GENE_NL_ECUDA;
    return GENE_NL_OK;
}

int gene_nl_compute_em(gene_nl_plan* h, const void* phi_, const void* apar_, const double* vpar_host,
                       const void* g_, void* rhs_, double scale, void* stream)
{
    g_err.clear();
    if (!h) { set_err("NULL plan"); return GENE_NL_EINVAL; }
    if (!h->em) { set_err("gene_nl_compute_em needs a plan created with chi_has_v = GENE_NL_CHI_EM"); return GENE_NL_EINVAL; }
    if (!vpar_host) { set_err("NULL v_par array"); return GENE_NL_EINVAL; }
    if (!on_plan_device(h)) return GENE_NL_EINVAL;
    if (!h->scr.Z) { set_err("the plan has no scratch (an earlier gene_nl_set_scratch_bytes ran out of memory)"); return GENE_NL_ENOMEM; }
    const size_t gbytes = sizeof(cplx) * h->M * (size_t)h->planes;
    const size_t cbytes = gbytes / h->nv;
    int rc = check_ptrs(phi_, g_, rhs_, gbytes, cbytes);
    if (!rc) rc = check_ptrs(apar_, g_, rhs_, gbytes, cbytes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone) {
        // (the host wait on the pinned v_par staging buffer would invalidate the capture)
        set_err("gene_nl_compute_em cannot be captured in a CUDA graph (host-side staging of v_par); gene_nl_compute can");
        return GENE_NL_EUNSUPPORTED;
    }
    cudaGetLastError();
    rc = stage_vpar(h, vpar_host, st);
    if (rc) return rc;
    if (enqueue_slabs(h, h->scr, (const cplx*)phi_, (const cplx*)g_, (cplx*)rhs_, h->nw * h->nspec, scale, st, nullptr,
                      (const cplx*)apar_) < 0)
        return GENE_NL_ECUDA;
    return GENE_NL_OK;
}

int gene_nl_compute(gene_nl_plan* h, const void* chi, const void* g, void* rhs, double scale, void* stream)
{
    return compute_impl(h, chi, g, rhs, scale, stream, nullptr);
}

int gene_nl_compute_profiled(gene_nl_plan* h, const void* chi, const void* g, void* rhs, double scale, void* stream,
                             double* ms4, int* launches4)  /* arrays of GENE_NL_KERNEL_CLASSES entries */
{
    if (!ms4 || !launches4) { set_err("NULL output pointer"); return GENE_NL_EINVAL; }
    Profiler prof;
    prof.st = (cudaStream_t)stream;
    int rc = compute_impl(h, chi, g, rhs, scale, stream, &prof);
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
    for (int c = 0; c < K_CLASSES; ++c) { ms4[c] = 0.0; launches4[c] = 0; }
    for (size_t i = 0; i < prof.cls.size(); ++i) {
        float ms = 0.f;
        if (e == cudaSuccess && cudaEventElapsedTime(&ms, prof.ev[2 * i], prof.ev[2 * i + 1]) == cudaSuccess) {
            ms4[prof.cls[i]] += ms;
            launches4[prof.cls[i]] += 1;
        }
    }
    for (auto ev : prof.ev) cudaEventDestroy(ev);
    if (rc) return rc;
    return cuda_ok(e, "cudaStreamSynchronize") ? GENE_NL_OK : GENE_NL_ECUDA;
}

// Host streaming: one chunk = one (w,s) slab = nz*nv contiguous planes of g and rhs and nz (or nz*nv)
// planes of chi (em: nz planes of phi_bar and of A_par_bar); three stages, each with its own stream, staging buffers
// and scratch set sized for ONE slab, so that the copies of one slab overlap the kernels of another.
static int host_impl(gene_nl_plan* h, const void* chi_, const void* apar_, const void* g_, void* rhs_, double scale)
{
    const size_t gbytes = sizeof(cplx) * h->M * (size_t)h->planes;
    const size_t cbytes = h->chi_has_v ? gbytes : gbytes / h->nv;
    int rc = check_ptrs(chi_, g_, rhs_, gbytes, cbytes);
    if (!rc && apar_) rc = check_ptrs(apar_, g_, rhs_, gbytes, cbytes);
    if (rc) return rc;
    const size_t slab_g = sizeof(cplx) * h->M * (size_t)h->nz * h->nv;
    const size_t slab_c = h->chi_has_v ? slab_g : slab_g / h->nv;
    if (h->stages.empty()) {
        // built locally and moved into the plan only when every allocation succeeded
        const int nstage = 3;
        std::vector<HostStage> st(nstage);
        size_t rbytes1 = h->rbytes;  // a stage's scratch set serves ONE slab: its real-space chi fields (em: of both
        if (h->fused)                // potentials; chi through the plane kernel: none), not those of a launch of nss slabs
            rbytes1 = h->fk.chiv ? 256 : sizeof(cplx) * (size_t)h->Nx * h->Ny * (size_t)h->nz * (h->chi_has_v ? h->nv : 1) * (h->em ? 2 : 1);
        bool ok = true;
        for (auto& s : st) {
            ok = ok && cuda_ok(cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking), "cudaStreamCreate") &&
                 cuda_ok(cudaMalloc(&s.g, slab_g), "cudaMalloc(stage g)") &&
                 cuda_ok(cudaMalloc(&s.rhs, slab_g), "cudaMalloc(stage rhs)") &&
                 cuda_ok(cudaMalloc(&s.chi, slab_c), "cudaMalloc(stage chi)") &&
                 (!h->em || cuda_ok(cudaMalloc(&s.apar, slab_c), "cudaMalloc(stage A_par)")) &&
                 alloc_scratch(h->zbytes, h->pbytes, rbytes1, &s.scr) && alloc_group_scratch(h, &s.scr);
            if (!ok) break;
        }
        if (!ok) {
            std::string keep = g_err;
            for (auto& s : st) {
                cudaFree(s.g); cudaFree(s.rhs); cudaFree(s.chi); cudaFree(s.apar);
                free_scratch(&s.scr);
                if (s.stream) cudaStreamDestroy(s.stream);
            }
            g_err = keep;
            return GENE_NL_ENOMEM;
        }
        h->stages = std::move(st);
    }
    const char* chi = (const char*)chi_;
    const char* apar = (const char*)apar_;
    const char* g = (const char*)g_;
    char* rhs = (char*)rhs_;
    int ret = GENE_NL_OK;
    for (int ws = 0; ws < h->nw * h->nspec && ret == GENE_NL_OK; ++ws) {
        HostStage& s = h->stages[ws % h->stages.size()];
        bool ok = cuda_ok(cudaMemcpyAsync(s.g, g + ws * slab_g, slab_g, cudaMemcpyHostToDevice, s.stream), "H2D g") &&
                  cuda_ok(cudaMemcpyAsync(s.rhs, rhs + ws * slab_g, slab_g, cudaMemcpyHostToDevice, s.stream), "H2D rhs") &&
                  cuda_ok(cudaMemcpyAsync(s.chi, chi + ws * slab_c, slab_c, cudaMemcpyHostToDevice, s.stream), "H2D chi") &&
                  (!apar || cuda_ok(cudaMemcpyAsync(s.apar, apar + ws * slab_c, slab_c, cudaMemcpyHostToDevice, s.stream), "H2D A_par"));
        if (!ok) { ret = GENE_NL_ECUDA; break; }
        if (enqueue_slabs(h, s.scr, s.chi, s.g, s.rhs, 1, scale, s.stream, nullptr, apar ? s.apar : nullptr, ws) < 0) { ret = GENE_NL_ECUDA; break; }
        if (!cuda_ok(cudaMemcpyAsync(rhs + ws * slab_g, s.rhs, slab_g, cudaMemcpyDeviceToHost, s.stream), "D2H rhs")) ret = GENE_NL_ECUDA;
    }
    for (auto& s : h->stages)
        if (!cuda_ok(cudaStreamSynchronize(s.stream), "cudaStreamSynchronize") && ret == GENE_NL_OK) ret = GENE_NL_ECUDA;
    return ret;
}

int gene_nl_compute_host(gene_nl_plan* h, const void* chi_, const void* g_, void* rhs_, double scale)
{
    g_err.clear();
    if (!h) { set_err("NULL plan"); return GENE_NL_EINVAL; }
    if (h->em) { set_err("plan was created with GENE_NL_CHI_EM: call gene_nl_compute_em_host"); return GENE_NL_EINVAL; }
    if (!on_plan_device(h)) return GENE_NL_EINVAL;
    return host_impl(h, chi_, nullptr, g_, rhs_, scale);
}

int gene_nl_compute_em_host(gene_nl_plan* h, const void* phi_, const void* apar_, const double* vpar_host, const void* g_,
                            void* rhs_, double scale)
{
    g_err.clear();
    if (!h) { set_err("NULL plan"); return GENE_NL_EINVAL; }
    if (!h->em) { set_err("gene_nl_compute_em_host needs a plan created with chi_has_v = GENE_NL_CHI_EM"); return GENE_NL_EINVAL; }
    if (!vpar_host || !apar_) { set_err("NULL v_par or A_par array"); return GENE_NL_EINVAL; }
    if (!on_plan_device(h)) return GENE_NL_EINVAL;
    // v_par reaches the device before any stage starts (legacy default stream + a device-wide wait is simplest and
    // happens once per call)
    int rc = stage_vpar(h, vpar_host, nullptr);
    if (rc) return rc;
    if (!cuda_ok(cudaEventSynchronize(h->vp_event), "cudaEventSynchronize(v_par)")) return GENE_NL_ECUDA;
    return host_impl(h, phi_, apar_, g_, rhs_, scale);
}

size_t gene_nl_workspace_bytes(const gene_nl_plan* h)
{
    if (!h) return 0;
    size_t n = h->zbytes + h->pbytes + h->rbytes + h->table_bytes;
    if (h->fused && h->fk.fng) {   // the group kernel's L2-resident scratch and its hand-over counters
        const size_t ngroup = (size_t)(h->fused_grid / h->fk.group);
        n += h->fk.group_scratch * ngroup + sizeof(unsigned) * 2 * ngroup;
    }
    if (h->em) n += sizeof(double) * (size_t)h->nv * h->nspec;
    return n;
}

int gene_nl_launches_per_compute(const gene_nl_plan* h)
{
    if (!h) return 0;
    const int nslab = h->nw * h->nspec;
    if (h->fused) {
        int n = 0;
        const size_t cps = (size_t)h->nz * (h->chi_has_v ? h->nv : 1);
        for (int s0 = 0; s0 < nslab; s0 += h->nss) {
            const int ns = (nslab - s0 < h->nss) ? nslab - s0 : h->nss;
            n += (h->fk.chiv ? 0 : (h->em ? 4 : 2) * (int)((cps * ns + (size_t)h->nbz - 1) / (size_t)h->nbz)) + 1;
        }
        return n;
    }
    return nslab * chunks_per_slab(h) * launches_per_chunk(h);
}

double gene_nl_query(const gene_nl_plan* h, int what)
{
    if (!h) return NAN;
    const double c = h->chi_has_v ? 1.0 : (h->em ? 2.0 : 1.0) / h->nv;  // em: two chi-like fields per (z,w,s)
    const double M = (double)h->M, Nx = h->Nx, Ny = h->Ny;
    switch (what) {
    case 0: return (double)h->planes;
    case 1: return Nx;
    case 2: return Ny;
    case 3: return h->fused ? (double)h->nss * h->nz * h->nv : (double)h->nzb * h->nvb;
    case 4: return h->fused ? (double)((h->nw * h->nspec + h->nss - 1) / h->nss)
                            : (double)h->nw * h->nspec * chunks_per_slab(h) * ((h->nv + h->nvb - 1) / h->nvb);
    case 7: return h->fused ? 1.0 : 0.0;
    case 8: return h->fk.fnc ? 1.0 : (h->fk.fng ? (h->fk.wa ? 4.0 : 2.0) : 0.0);
    case 5: return 16.0 * M * (3.0 + c);
    case 6: {
        const double t2d = h->nky0 * 5.0 * Nx * std::log2(Nx) + Nx * 2.5 * Ny * std::log2(Ny);
        return (3.0 + 2.0 * c) * t2d + 4.0 * M * (1.0 + c) + (h->em ? 7.0 : 3.0) * Nx * Ny + 4.0 * M;  // em: +2 FMA/point
    }
    default: return NAN;
    }
}

}  // extern "C"
