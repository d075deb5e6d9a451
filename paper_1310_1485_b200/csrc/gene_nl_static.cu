// gene_nl_static.cu -- gene_nl_compute_static (include/gene_nl.h): the E x B term for callers that must not allocate.
//
// Who this is for.  Everything else in this library works through a plan, and gene_nl_create / gene_nl_compute_host /
// gene_nl_set_* call cudaMalloc (tables, the Z / P / R scratch, staging buffers).  Three kinds of caller cannot use that:
//   * a simulation that hands ALL device memory to its own pool allocator at start-up (a 180 GB B200 filled with
//     distribution functions): a later cudaMalloc inside a library simply fails;
//   * a time-step loop that runs next to other streams (halo exchange, diagnostics): cudaMalloc and cudaFree
//     synchronise the whole device and would stall them;
//   * code that runs where the CUDA runtime forbids allocation, e.g. between cudaStreamBeginCapture and EndCapture
//     of somebody else's graph.
// For them there is this ONE entry point.  It takes no plan; the caller passes the inputs and the output, and the only
// other global memory the kernel touches is file-scope `static __device__` storage of this translation unit:
//   s_scratch   kStaticGroups slots of Z(g) + Z(chi) + P, 552 960 B each: the half-transformed plane of every group of
//               the persistent kernel (the "transposed" intermediate of PAPER.md:61), 33.75 MiB in all;
//   s_cnt       two hand-over counters per group;
//   s_tables    the root tables W_144^k for the x and the y transforms (4.5 KiB).
// Every GPU whose context loads libgene_nl.so holds these 33.8 MiB from the load to the end of the process, whether or
// not this entry point is ever called: that is the price, and the reason the maximum is kept modest (64 planes in
// flight: 64 of the 148 SMs of a B200 work; gene_nl_compute with a plan uses them all).
//
// The kernel is one more instantiation of the group kernel of nl_group.cuh (groups of ONE CTA, 144 x 144 padded grid,
// chi per plane, the operator of BASELINE.json configs[4]): same phases, same arithmetic, but handed the address of the
// static scratch instead of a cudaMalloc'ed one.  In HOST code the name `s_scratch` is only a stand-in symbol, not a
// device address: the address comes from cudaGetSymbolAddress, once per device and with that device current
// (setup_device below).  Passing the bare name to the kernel would hand it a host pointer.
//
// Sharing.  All calls on a device use the same array and find in it whatever the previous call left.  Nothing in Z or P
// has to start at zero (each plane writes every slot of its group's Z before the y phase reads it, and every slot of P
// before the x-analysis reads it); the counters do, and are cleared on the caller's stream before every launch.  Two
// calls that overlap on the GPU (different streams, or different host threads on the same device) would write the same
// slots: they RACE.  Keep calls on one device in one stream, or order them with events.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include <string>

#include "../../include/gene_nl.h"
#include "nl_group.cuh"

using gnl::cplx;

extern "C" void gene_nl_set_error_(const char* msg);  // gene_nl.cu: the thread-local string of gene_nl_last_error

namespace {

// 144 x 144 padded grid = 12 x 12 (x) by 18 x 8 (y), groups of one CTA of 8 warps, chi per plane.  AX2 / BX2 are given
// explicitly (the same split as the synthesis): that makes this a symbol of its own, distinct from the instantiation
// gene_nl.cu launches for plans, so nothing the plan path configures or launches is shared with it.
using KS = gnl::Grouped<12, 12, 18, 1, 8, 1, true, 8, 3, 12, 12, 8>;
#define GNL_STATIC_KERNEL gnl::k_plane_group<12, 12, 18, 1, 8, 1, true, false, 8, 3, 12, 12, 8>

constexpr int kStaticGroups = GENE_NL_STATIC_MAX_GROUPS;            // slots = planes in flight
constexpr size_t kSlotCplx = KS::GROUP_SCRATCH_CPLX;                // 2 * 13 824 (Z of g and chi) + 6 912 (P) values
constexpr int kMaxDevices = 64;
static_assert(KS::NX == 144 && KS::NY == 144 && KS::NX0 == GENE_NL_STATIC_NX0 && KS::NKY0 == GENE_NL_STATIC_NKY0, "the one supported grid");
static_assert(kSlotCplx * sizeof(cplx) == 552960, "slot size quoted in include/gene_nl.h and README.md");
static_assert(KS::SMEM_BYTES <= 227 * 1024, "one CTA per SM");

// The scratch.  Device code of this file could name these arrays directly; host code needs cudaGetSymbolAddress.
static __device__ __align__(256) cplx s_scratch[(size_t)kStaticGroups * kSlotCplx];
static __device__ __align__(256) unsigned s_cnt[2 * kStaticGroups];
static __device__ __align__(256) cplx s_tables[KS::NX + KS::NY];

struct DeviceState {
    bool ready = false;
    cplx* scratch = nullptr;   // device address of s_scratch on this device
    unsigned* cnt = nullptr;   // ... of s_cnt
    cplx* tables = nullptr;    // ... of s_tables: W_NX^k, then W_NY^k
    int groups = 0;            // CTAs the device keeps resident, at most kStaticGroups
};
DeviceState g_state[kMaxDevices];
std::mutex g_mutex;

bool ok_or_err(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return true;
    gene_nl_set_error_((std::string("gene_nl_compute_static: ") + what + ": " + cudaGetErrorString(e)).c_str());
    return false;
}

// Once per device, with that device current: addresses of the static arrays, the root tables, the kernel's shared-memory
// limit, the grid.  Uses a synchronous copy, so it must not happen inside a stream capture (see the header).
bool setup_device(int dev, DeviceState* st)
{
    cplx *scratch = nullptr, *tables = nullptr;
    unsigned* cnt = nullptr;
    if (!ok_or_err(cudaGetSymbolAddress((void**)&scratch, s_scratch), "cudaGetSymbolAddress(scratch)") ||
        !ok_or_err(cudaGetSymbolAddress((void**)&cnt, s_cnt), "cudaGetSymbolAddress(counters)") ||
        !ok_or_err(cudaGetSymbolAddress((void**)&tables, s_tables), "cudaGetSymbolAddress(tables)"))
        return false;
    cplx host_tab[KS::NX + KS::NY];   // on the stack: no allocation of any kind
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int k = 0; k < KS::NX; ++k) {
        const long double a = two_pi * (long double)k / (long double)KS::NX;
        host_tab[k].x = (double)cosl(a);
        host_tab[k].y = (double)sinl(a);
    }
    for (int k = 0; k < KS::NY; ++k) {
        const long double a = two_pi * (long double)k / (long double)KS::NY;
        host_tab[KS::NX + k].x = (double)cosl(a);
        host_tab[KS::NX + k].y = (double)sinl(a);
    }
    if (!ok_or_err(cudaMemcpy(tables, host_tab, sizeof host_tab, cudaMemcpyHostToDevice), "cudaMemcpy(root tables)")) return false;
    if (!ok_or_err(cudaFuncSetAttribute(GNL_STATIC_KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)KS::SMEM_BYTES),
                   "cudaFuncSetAttribute(shared memory)"))
        return false;
    int sms = 0, occ = 0;
    if (!ok_or_err(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute") ||
        !ok_or_err(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, GNL_STATIC_KERNEL, KS::NT, KS::SMEM_BYTES), "occupancy query"))
        return false;
    if (sms < 1 || occ < 1) {
        gene_nl_set_error_("gene_nl_compute_static: the kernel does not fit an SM of this device");
        return false;
    }
    st->scratch = scratch;
    st->cnt = cnt;
    st->tables = tables;
    st->groups = sms * occ < kStaticGroups ? sms * occ : kStaticGroups;
    st->ready = true;
    return true;
}

}  // namespace

extern "C" int gene_nl_compute_static(int nx0, int nky0, int nz, int nv, int nw, int nspec, double kxmin, double kymin,
                                      const void* chi_, const void* g_, void* rhs_, double scale, void* stream)
{
    gene_nl_set_error_("");
    if (nz <= 0 || nv <= 0 || nw <= 0 || nspec <= 0 || !std::isfinite(kxmin) || !std::isfinite(kymin)) {
        gene_nl_set_error_("gene_nl_compute_static: extents must be positive, kxmin/kymin finite");
        return GENE_NL_EINVAL;
    }
    if (nx0 != GENE_NL_STATIC_NX0 || nky0 != GENE_NL_STATIC_NKY0) {
        char buf[320];
        snprintf(buf, sizeof buf,
                 "gene_nl_compute_static: %d x %d modes per plane, but the static scratch is laid out for planes of exactly %d x %d "
                 "modes (552960 B per plane in flight, %d planes in flight); other sizes need a plan (gene_nl_create), which allocates",
                 nx0, nky0, GENE_NL_STATIC_NX0, GENE_NL_STATIC_NKY0, kStaticGroups);
        gene_nl_set_error_(buf);
        return GENE_NL_EUNSUPPORTED;
    }
    const long long planes = (long long)nz * nv * nw * nspec;
    if ((long long)nz * nv > GENE_NL_STATIC_MAX_PLANES || (long long)nw * nspec > GENE_NL_STATIC_MAX_PLANES || planes > GENE_NL_STATIC_MAX_PLANES) {
        gene_nl_set_error_("gene_nl_compute_static: more than GENE_NL_STATIC_MAX_PLANES (2^31 - 1) planes in one call: split the call");
        return GENE_NL_EUNSUPPORTED;
    }
    if (!chi_ || !g_ || !rhs_) { gene_nl_set_error_("gene_nl_compute_static: NULL array pointer"); return GENE_NL_EINVAL; }
    if (((uintptr_t)chi_ | (uintptr_t)g_ | (uintptr_t)rhs_) & 15) {
        gene_nl_set_error_("gene_nl_compute_static: array pointers must be 16-byte aligned");
        return GENE_NL_EINVAL;
    }
    const size_t bytes = sizeof(cplx) * (size_t)nx0 * nky0 * (size_t)planes;
    const char *r0 = (const char*)rhs_, *g0 = (const char*)g_, *c0 = (const char*)chi_;
    if ((g0 < r0 + bytes && r0 < g0 + bytes) || (c0 < r0 + bytes && r0 < c0 + bytes)) {
        gene_nl_set_error_("gene_nl_compute_static: rhs overlaps g or chi");
        return GENE_NL_EINVAL;
    }
    int dev = -1;
    if (!ok_or_err(cudaGetDevice(&dev), "cudaGetDevice (no CUDA device: this library has no CPU fallback)")) return GENE_NL_ECUDA;
    if (dev < 0 || dev >= kMaxDevices) { gene_nl_set_error_("gene_nl_compute_static: device ordinal beyond 63"); return GENE_NL_EUNSUPPORTED; }
    DeviceState st;
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!g_state[dev].ready && !setup_device(dev, &g_state[dev])) return GENE_NL_ECUDA;
        st = g_state[dev];
    }
    cudaStream_t s = (cudaStream_t)stream;
    const int grid = planes < st.groups ? (int)planes : st.groups;
    // the counters start every launch at zero (groups of one CTA order their phases by the CTA barrier and leave them
    // alone; cleared all the same, as the kernel's contract asks)
    if (!ok_or_err(cudaMemsetAsync(st.cnt, 0, sizeof(unsigned) * 2 * kStaticGroups, s), "cudaMemsetAsync(counters)")) return GENE_NL_ECUDA;
    const double coef = scale / (2.0 * (double)KS::NX * (double)KS::NY);
    GNL_STATIC_KERNEL<<<grid, KS::NT, KS::SMEM_BYTES, s>>>(
        (const cplx*)g_, (cplx*)rhs_, (const cplx*)nullptr, (const cplx*)chi_, (const cplx*)st.tables,
        (const cplx*)(st.tables + KS::NX), st.scratch, st.cnt, nz, nv, nw * nspec, kxmin, kymin, coef,
        (const cplx*)nullptr, (const double*)nullptr, nw, 0);
    if (!ok_or_err(cudaGetLastError(), "kernel launch")) return GENE_NL_ECUDA;
    return GENE_NL_OK;
}
