// gene_nlx.cu -- C ABI of the x-global nonlinearity (include/gene_nl.h, gene_nlx_*): plan, launch.
// One kernel (nlx_kernel.cuh) per compute; nothing but the twiddle table lives in the plan.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>

#include "../../include/gene_nl.h"
#include "nlx_kernel.cuh"

using gnl::cplx;

extern "C" void gene_nl_set_error_(const char* msg);  // gene_nl.cu: the thread-local string of gene_nl_last_error

namespace {

typedef void (*xg_fn)(const cplx*, const cplx*, const cplx*, const cplx*, const double*, cplx*, const cplx*, int, int,
                      long long, double);
struct XgKernel {
    xg_fn fn = nullptr;
    size_t smem = 0;
    int nt = 0, xt = 32;  // threads per CTA, x points per tile
};
template <int NY, int A, int B, int NT, int XT = 32>
XgKernel make_xg()
{
    XgKernel k;
    k.fn = gnl::k_xglobal<NY, A, B, NT, XT>;
    k.smem = gnl::XGlobal<NY, A, B, NT, XT>::SMEM_BYTES;
    k.nt = NT;
    k.xt = XT;
    return k;
}
bool find_xg(int ny, XgKernel* out)
{
    switch (ny) {
    // 16 x points per tile and 64 threads: 5 CTAs per SM at Ny = 48 (measured on B200: 42.6 M planes/s against 37.4
    // with 32 x points and 128 threads)
    case 24: *out = make_xg<24, 3, 8, 64, 16>(); return true;
    case 48: *out = make_xg<48, 6, 8, 64, 16>(); return true;   // the paper's 64 x 16 planes
    case 96: *out = make_xg<96, 12, 8, 64, 16>(); return true;
    // longer y grids (not the paper's size): 8 x points per tile so that the staging and exchange tiles fit beside each other
    case 144: *out = make_xg<144, 18, 8, 64, 8>(); return true;
    case 192: *out = make_xg<192, 24, 8, 64, 8>(); return true;
    case 288: *out = make_xg<288, 18, 16, 64, 8>(); return true;
    case 384: *out = make_xg<384, 24, 16, 64, 8>(); return true;
    default: return false;
    }
}

bool ok_or_err(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return true;
    gene_nl_set_error_((std::string(what) + ": " + cudaGetErrorString(e)).c_str());
    return false;
}

}  // namespace

struct XgStage {  // per-stream staging of one chunk of planes for gene_nlx_compute_host
    cudaStream_t stream = nullptr;
    cplx* buf[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};  // vex, vey, dxg, dyg, rhs
};

struct gene_nlx_plan {
    int nx, nky0, Ny;
    long long planes;
    XgKernel k;
    cplx* tw = nullptr;
    int grid_cap = 0;
    int device = -1;
    std::vector<XgStage> stages;  // lazily created by gene_nlx_compute_host
    long long chunk = 0;          // planes per chunk
    double* pref_dev = nullptr;
};

extern "C" {

gene_nlx_plan* gene_nlx_create(int nx, int nky0, long long planes)
{
    gene_nl_set_error_("");
    if (nx <= 0 || nky0 <= 0 || planes <= 0) {
        gene_nl_set_error_("gene_nlx_create: extents must be positive");
        return nullptr;
    }
    int dev = -1;
    if (!ok_or_err(cudaGetDevice(&dev), "cudaGetDevice (no CUDA device: this library has no CPU fallback)")) return nullptr;
    gene_nlx_plan* h = new gene_nlx_plan();
    h->nx = nx; h->nky0 = nky0; h->Ny = 3 * nky0; h->planes = planes; h->device = dev;
    if (!find_xg(h->Ny, &h->k)) {
        gene_nl_set_error_("gene_nlx_create: unsupported nky0 (padded y grid Ny = 3 nky0 must be 24, 48, 96, 144, 192, 288 or 384)");
        delete h;
        return nullptr;
    }
    std::vector<cplx> t(h->Ny);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int k = 0; k < h->Ny; ++k) {
        const long double ang = two_pi * (long double)k / (long double)h->Ny;
        t[k].x = (double)cosl(ang);
        t[k].y = (double)sinl(ang);
    }
    int sms = 0, occ = 0;
    bool ok = ok_or_err(cudaMalloc(&h->tw, sizeof(cplx) * h->Ny), "cudaMalloc(twiddles)") &&
              ok_or_err(cudaMemcpy(h->tw, t.data(), sizeof(cplx) * h->Ny, cudaMemcpyHostToDevice), "cudaMemcpy(twiddles)") &&
              ok_or_err(cudaFuncSetAttribute(h->k.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->k.smem), "k_xglobal smem") &&
              ok_or_err(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute") &&
              ok_or_err(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, h->k.fn, h->k.nt, h->k.smem), "occupancy(k_xglobal)");
    if (!ok || occ < 1) {
        if (ok) gene_nl_set_error_("k_xglobal does not fit on an SM");
        gene_nlx_destroy(h);
        return nullptr;
    }
    h->grid_cap = occ * sms * 8;  // grid-stride over the tiles, a few CTAs per resident slot
    return h;
}

static int check_args(const gene_nlx_plan* h, const void* vex, const void* vey, const void* dxg, const void* dyg,
                      const double* pref, const void* rhs)
{
    if (!h) { gene_nl_set_error_("NULL plan"); return GENE_NL_EINVAL; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) {
        gene_nl_set_error_("the current CUDA device is not the one the plan was created on");
        return GENE_NL_EINVAL;
    }
    if (!vex || !vey || !dxg || !dyg || !pref || !rhs) { gene_nl_set_error_("NULL array pointer"); return GENE_NL_EINVAL; }
    if (((uintptr_t)vex | (uintptr_t)vey | (uintptr_t)dxg | (uintptr_t)dyg | (uintptr_t)rhs) & 15) {
        gene_nl_set_error_("array pointers must be 16-byte aligned");
        return GENE_NL_EINVAL;
    }
    const size_t bytes = sizeof(cplx) * (size_t)h->nx * h->nky0 * (size_t)h->planes;
    const char* r0 = (const char*)rhs;
    for (const void* in : {vex, vey, dxg, dyg}) {
        const char* a = (const char*)in;
        if (a < r0 + bytes && r0 < a + bytes) { gene_nl_set_error_("rhs overlaps an input array"); return GENE_NL_EINVAL; }
    }
    return GENE_NL_OK;
}

// one launch of k_xglobal over `planes` planes starting at the given device pointers
static bool launch(const gene_nlx_plan* h, const cplx* vex, const cplx* vey, const cplx* dxg, const cplx* dyg,
                   const double* pref, cplx* rhs, long long planes, double scale, cudaStream_t st)
{
    const int xtiles = (h->nx + h->k.xt - 1) / h->k.xt;
    const long long ntiles = planes * xtiles;
    const int grid = (int)(ntiles < h->grid_cap ? ntiles : h->grid_cap);
    const double coef = scale / (2.0 * (double)h->Ny);
    h->k.fn<<<grid, h->k.nt, h->k.smem, st>>>(vex, vey, dxg, dyg, pref, rhs, h->tw, h->nx, xtiles, ntiles, coef);
    return ok_or_err(cudaGetLastError(), "k_xglobal launch");
}

int gene_nlx_compute(gene_nlx_plan* h, const void* vex, const void* vey, const void* dxg, const void* dyg,
                     const double* pref, void* rhs, double scale, void* stream)
{
    gene_nl_set_error_("");
    const int rc = check_args(h, vex, vey, dxg, dyg, pref, rhs);
    if (rc) return rc;
    return launch(h, (const cplx*)vex, (const cplx*)vey, (const cplx*)dxg, (const cplx*)dyg, pref, (cplx*)rhs, h->planes,
                  scale, (cudaStream_t)stream) ? GENE_NL_OK : GENE_NL_ECUDA;
}

static void free_xg_stages(gene_nlx_plan* h)
{
    for (auto& s : h->stages) {
        for (cplx* b : s.buf) cudaFree(b);
        if (s.stream) cudaStreamDestroy(s.stream);
    }
    h->stages.clear();
    cudaFree(h->pref_dev);
    h->pref_dev = nullptr;
}

// "we split each input array into (usually four) contiguous chunks of xy-planes, which are transferred
// and computed in two asynchronous CUDA streams".  Here: chunks of <= 64 MiB per array (at least four per call when
// the arrays allow it), three streams, so that the H2D copies of one chunk, the kernel of another and the D2H copy of
// a third overlap; 5 planes go in and 1 comes out per plane computed.
int gene_nlx_compute_host(gene_nlx_plan* h, const void* vex, const void* vey, const void* dxg, const void* dyg,
                          const double* pref, void* rhs, double scale)
{
    gene_nl_set_error_("");
    const int rc = check_args(h, vex, vey, dxg, dyg, pref, rhs);
    if (rc) return rc;
    const size_t plane_bytes = sizeof(cplx) * (size_t)h->nx * h->nky0;
    if (h->stages.empty()) {
        long long chunk = (long long)(((size_t)64 << 20) / plane_bytes);
        if (chunk > (h->planes + 3) / 4) chunk = (h->planes + 3) / 4;
        if (chunk < 1) chunk = 1;
        std::vector<XgStage> st(3);
        bool ok = ok_or_err(cudaMalloc(&h->pref_dev, sizeof(double) * h->nx), "cudaMalloc(pref)");
        for (auto& s : st) {
            ok = ok && ok_or_err(cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking), "cudaStreamCreate");
            for (auto& b : s.buf) ok = ok && ok_or_err(cudaMalloc(&b, plane_bytes * (size_t)chunk), "cudaMalloc(stage)");
            if (!ok) break;
        }
        h->stages = std::move(st);
        if (!ok) { free_xg_stages(h); return GENE_NL_ENOMEM; }
        h->chunk = chunk;
    }
    if (!ok_or_err(cudaMemcpy(h->pref_dev, pref, sizeof(double) * h->nx, cudaMemcpyHostToDevice), "cudaMemcpy(pref)"))
        return GENE_NL_ECUDA;
    const char* in[4] = {(const char*)vex, (const char*)vey, (const char*)dxg, (const char*)dyg};
    char* out = (char*)rhs;
    int ret = GENE_NL_OK;
    long long c = 0;
    for (long long p0 = 0; p0 < h->planes && ret == GENE_NL_OK; p0 += h->chunk, ++c) {
        XgStage& s = h->stages[c % h->stages.size()];
        const long long np = (h->planes - p0 < h->chunk) ? h->planes - p0 : h->chunk;
        const size_t off = plane_bytes * (size_t)p0, nb = plane_bytes * (size_t)np;
        bool ok = true;
        for (int a = 0; a < 4; ++a) ok = ok && ok_or_err(cudaMemcpyAsync(s.buf[a], in[a] + off, nb, cudaMemcpyHostToDevice, s.stream), "H2D");
        ok = ok && ok_or_err(cudaMemcpyAsync(s.buf[4], out + off, nb, cudaMemcpyHostToDevice, s.stream), "H2D rhs") &&
             launch(h, s.buf[0], s.buf[1], s.buf[2], s.buf[3], h->pref_dev, s.buf[4], np, scale, s.stream) &&
             ok_or_err(cudaMemcpyAsync(out + off, s.buf[4], nb, cudaMemcpyDeviceToHost, s.stream), "D2H rhs");
        if (!ok) ret = GENE_NL_ECUDA;
    }
    for (auto& s : h->stages)
        if (!ok_or_err(cudaStreamSynchronize(s.stream), "cudaStreamSynchronize") && ret == GENE_NL_OK) ret = GENE_NL_ECUDA;
    return ret;
}

void gene_nlx_destroy(gene_nlx_plan* h)
{
    if (!h) return;
    cudaDeviceSynchronize();
    free_xg_stages(h);
    cudaFree(h->tw);
    delete h;
}

double gene_nlx_query(const gene_nlx_plan* h, int what)
{
    if (!h) return NAN;
    const double M = (double)h->nx * h->nky0, Ny = h->Ny;
    switch (what) {
    case 0: return (double)h->planes;
    case 1: return Ny;
    case 5: return 16.0 * M * 6.0;  // 5 planes read, 1 written ("5 input, 1 output")
    case 6: return h->nx * (5.0 * 2.5 * Ny * std::log2(Ny) + 3.0 * Ny) + 4.0 * M;  // 4 c2r + 1 r2c, multiply, prefactor+add
    default: return NAN;
    }
}

}  // extern "C"
