/*
 * gene_nl.h -- C ABI of the B200-native E x B nonlinearity of GENE (flux-tube, pseudo-spectral).
 *
 * Operation (sect. 2.1; operator/layout per BASELINE.json north_star):
 * for every (z, v_par, mu, species) plane p
 *
 *     rhs[:, :, p] += scale * N(chi_p, g_p),
 *     N = dx(chi) * dy(g) - dy(chi) * dx(g)          (the E x B bracket, dealiased by the 3/2 rule)
 *
 * i.e. "the fields are preprocessed (... extension ... for dealiasing according to the 3/2-rule)
 * ..., a fast Fourier transform to real space is applied.  After multiplication the result is
 * transformed back to the spectral representation, the additional modes are deleted, ... multiplied
 * with a prefactor, and is finally added to the right-hand side vector", with the
 * spectral derivatives i*kx, i*ky formed on the device from g and chi (north_star; the paper's
 * port received them pre-differentiated).  The result equals the truncated spectral
 * convolution  N(a,b) = sum_{k'+k''=k} (ky' kx'' - kx' ky'') chi(k') g(k'')  up to FP64 rounding.
 *
 * Layout (BASELINE.json configs[0]).  All arrays are complex128 (re, im interleaved doubles).
 *   g, rhs : extents [nx0, nky0, nz, nv, nw, nspec], kx fastest:
 *            offset(i,j,k,l,m,n) = i + nx0*(j + nky0*(k + nz*(l + nv*(m + nw*n)))).
 *   chi    : chi_has_v = 0 -> [nx0, nky0, nz, nw, nspec] (no v extent, broadcast over v);
 *            chi_has_v = 1 -> same extents as g.
 *   kx of row i: kxmin*i (i < nx0/2), kxmin*(i - nx0) (i > nx0/2).  Row i = nx0/2 (Nyquist) is
 *   ignored in chi and g and left untouched in rhs.  ky of column j: kymin*j, j = 0..nky0-1; the
 *   ky < 0 half is implied by reality.  The ky = 0 column should be Hermitian in kx; if it is not,
 *   its Hermitian part is used (the real part of the synthesis).
 *   Padded real grid: Nx = 3*nx0/2 by Ny = 3*nky0.
 *
 * Everything runs in hand-written sm_100a CUDA kernels in FP64.  There is no CPU fallback, no cuFFT,
 * no backend dispatch: on a machine without a CUDA device gene_nl_create fails.
 */
#ifndef GENE_NL_H
#define GENE_NL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gene_nl_plan gene_nl_plan; /* opaque */

/* error codes returned by gene_nl_compute* (0 = success) */
#define GENE_NL_OK 0
#define GENE_NL_EINVAL 1       /* NULL / misaligned / overlapping pointer, bad handle            */
#define GENE_NL_EUNSUPPORTED 2 /* grid size without an instantiated kernel                        */
#define GENE_NL_ECUDA 3        /* a CUDA runtime call or kernel launch failed                     */
#define GENE_NL_ENOMEM 4       /* device or pinned-host allocation failed                         */

/*
 * gene_nl_create -- build a plan on the CURRENT CUDA device (north_star signature).
 *   nx0   number of kx modes (even; Nx = 3*nx0/2 must be one of 24,48,96,144,192,288,384,576,768,1152,1536)
 *   nky0  number of ky >= 0 modes (Ny = 3*nky0 must be one of 24,48,96,144,192,288,384,576)
 *   nz, nv, nw, nspec   extents of the parametric dimensions (all > 0); planes = nz*nv*nw*nspec
 *   kxmin, kymin        wavenumber spacings (finite)
 *   chi_has_v           0: chi has no v extent (shared by the nv planes); 1: chi shaped like g
 * The plan owns its device tables and scratch (allocated here, freed by gene_nl_destroy).
 * Returns NULL on failure; gene_nl_last_error() then describes why.
 */
gene_nl_plan* gene_nl_create(int nx0, int nky0, int nz, int nv, int nw, int nspec,
                             double kxmin, double kymin, int chi_has_v);

/*
 * gene_nl_compute -- rhs += scale * N(chi, g) for all planes.  DEVICE pointers, caller-owned, 16-byte
 * aligned, layouts as above; chi and g are read-only, rhs must not overlap them.  `stream` is a
 * cudaStream_t passed as void* (NULL = legacy default stream).  Asynchronous: all work is enqueued on
 * `stream` and the call returns without synchronising.  One compute may be in flight per plan (the
 * scratch is shared).  Returns GENE_NL_OK or an error code; on error rhs may be partially updated.
 */
int gene_nl_compute(gene_nl_plan* h, const void* chi, const void* g, void* rhs, double scale,
                    void* stream);

/*
 * gene_nl_compute_em -- electromagnetic case with chi composed ON THE DEVICE (BASELINE.json
 * configs[4]: "phi - v_par*A_par is supplied per plane"; "moving more computation to the GPU, while
 * keeping the amount of transfer constant").  For a plan created with chi_has_v = GENE_NL_CHI_EM:
 *     rhs[.,.,p] += scale * N(chi_p, g_p),   chi_p = phi_bar[z,w,s] - vpar[v + nv*s] * apar_bar[z,w,s],  p = (z,v,w,s).
 * phi, apar: DEVICE arrays, complex128 [nx0, nky0, nz, nw, nspec] (the layout of chi without v); vpar: HOST array of
 * nv*nspec doubles, pageable or pinned: it is copied into a plan-owned pinned staging buffer before the call returns
 * (the caller may reuse it at once) and from there to the device on `stream`.  Because that staging buffer is reused,
 * a call first waits on the host for the previous call's copy, and the call is NOT capturable in a CUDA graph
 * (gene_nl_compute is).  By linearity the two fields are transformed to real space once per (z,w,s) and combined
 * inside the bracket kernel, so the per-plane chi array (as large as g) is never formed, read or transformed.  Other
 * arguments, errors and asynchrony as gene_nl_compute.  The group kernel composes chi where it exists (384 x 192 and
 * 144 x 144 padded grids), else the batched bracket kernel does.  Called while `stream` is being captured it returns
 * GENE_NL_EUNSUPPORTED and leaves the capture intact.  gene_nl_compute / gene_nl_compute_host reject such a plan.
 */
#define GENE_NL_CHI_EM 2
int gene_nl_compute_em(gene_nl_plan* h, const void* phi, const void* apar, const double* vpar_host, const void* g,
                       void* rhs, double scale, void* stream);

/* gene_nl_compute_em_host -- gene_nl_compute_em on HOST buffers (phi, apar, g, rhs; layouts as above), streamed through
 * the device one (w,s) slab at a time exactly as gene_nl_compute_host does.  SYNCHRONOUS. */
int gene_nl_compute_em_host(gene_nl_plan* h, const void* phi_host, const void* apar_host, const double* vpar_host,
                            const void* g_host, void* rhs_host, double scale);

/*
 * gene_nl_compute_host -- same operation on HOST buffers (same layouts).  The arrays are streamed
 * through the device in chunks of planes on several CUDA streams (one (w,s) slab each) so that host->device
 * copies, kernels and the device->host copy of rhs overlap ("we split each input array into
 * (usually four) contiguous chunks of xy-planes, which are transferred and computed in two
 * asynchronous CUDA streams").  Pinned (page-locked) host memory gives full overlap; pageable memory
 * works but copies serialise.  SYNCHRONOUS: returns after rhs_host holds the result.
 */
int gene_nl_compute_host(gene_nl_plan* h, const void* chi_host, const void* g_host, void* rhs_host,
                         double scale);

/* gene_nl_destroy -- free the plan's device memory.  NULL is a no-op.  Synchronises the device. */
void gene_nl_destroy(gene_nl_plan* h);

/* Thread-local description of the last failure in this library ("" if none). */
const char* gene_nl_last_error(void);

/* Bytes of device memory owned by the plan: root tables, the Z / P / R scratch set, the group kernel's per-group
 * scratch and hand-over counters, the v_par coefficients of an EM plan.  (The staging buffers the *_host entry points
 * create on first use are not counted.) */
size_t gene_nl_workspace_bytes(const gene_nl_plan* h);

/*
 * gene_nl_set_scratch_bytes -- change the plan's scratch budget (SURVEY.md 8(b) "optional workspace" extension).
 * The planes of one compute are walked in batches whose scratch (the half-transformed arrays Z and P and the
 * real-space chi fields) fits `bytes` per scratch set; the default is 768 MiB.  A smaller budget means more and
 * smaller launches (and ragged last batches), never a different result.  Synchronises the device, frees and
 * re-allocates the scratch (and drops the staging buffers of the host entry points).  bytes >= 1 MiB.
 * Returns GENE_NL_OK, or GENE_NL_ENOMEM with the previous budget restored.
 */
int gene_nl_set_scratch_bytes(gene_nl_plan* h, size_t bytes);

/* Number of kernel launches one gene_nl_compute enqueues (for launch accounting in benchmarks). */
int gene_nl_launches_per_compute(const gene_nl_plan* h);

/*
 * gene_nl_set_plane_kernel -- choose the kernel family for the g side of a plane.
 *   GENE_NL_KERNEL_AUTO     what gene_nl_create selected (the fastest measured on B200): the fused shared-memory kernel
 *                           for planes that fit one SM; beyond that the group kernel where it exists, else the batched
 *                           kernels.
 *   GENE_NL_KERNEL_GROUP    the fused kernel spread over groups of G co-resident CTAs (one cooperative launch, every SM
 *                           used): the two x<->y hand-overs of a plane (the "transpositions" of PAPER.md:61) go through
 *                           a per-group scratch that is rewritten every plane and therefore stays in L2; rows come
 *                           back by 1-D bulk copies (TMA).  HBM sees g, rhs and the chi rows only (1.02 - 1.46 x the
 *                           algorithmic bytes).  Exists, on a device with cooperative launch, for the padded grids
 *                             384 x 192 (nx0 = 256, nky0 = 64: configs[2])  G = 4, chi_has_v = 0 or GENE_NL_CHI_EM,
 *                             768 x 384 (nx0 = 512, nky0 = 128: configs[3]) G = 8, chi_has_v = 0,
 *                             144 x 144 (nx0 = 96, nky0 = 48: configs[4])   G = 1, chi_has_v = 0, 1 or GENE_NL_CHI_EM
 *                           (with chi_has_v = 1 chi goes through the same kernel: one launch per compute).
 *   GENE_NL_KERNEL_CLUSTER  the same phases over a thread-block cluster of 8 CTAs with the half-transformed plane in the
 *                           cluster's shared memory and distributed-shared-memory hand-overs (1.03 x the algorithmic
 *                           bytes; slower: DSMEM stores run at 18 B/clk/SM and 15 clusters fit the 148 SMs).  384 x 192
 *                           with chi_has_v = 0 only.
 *   GENE_NL_KERNEL_BATCHED  the batched kernels (scratch through HBM/L2 in large batches) whatever the size.
 *   GENE_NL_KERNEL_WARP     the group kernel with warp-autonomous x phases as well (a warp takes two adjacent columns
 *                           through both x stages in its own shared-memory tile; every warp arrives on the hand-over
 *                           counters; no CTA-wide barrier in the plane loop).  Measured on B200: 3 % faster than the
 *                           group kernel at 384 x 192, 10 % slower at 768 x 384 and 144 x 144 (DESIGN.md sect. 6g), so
 *                           it is an option, not the default.  384 x 192 and 768 x 384 with chi_has_v = 0, 144 x 144
 *                           with chi_has_v = 0 or 1; not with GENE_NL_CHI_EM.
 * GENE_NL_EUNSUPPORTED when the plan has no such kernel.  Same results to rounding (all are checked against the
 * oracle).  Synchronises the device and re-allocates the scratch, like gene_nl_set_scratch_bytes.
 */
#define GENE_NL_KERNEL_AUTO 0
#define GENE_NL_KERNEL_CLUSTER 1
#define GENE_NL_KERNEL_GROUP 2
#define GENE_NL_KERNEL_BATCHED 3
#define GENE_NL_KERNEL_WARP 4
int gene_nl_set_plane_kernel(gene_nl_plan* h, int kind);

/*
 * gene_nl_query -- plan facts for benchmarks and tests.  `what`:
 *   0 planes, 1 Nx, 2 Ny, 3 planes per batch, 4 batches per compute,
 *   5 algorithmic bytes per plane  B = 16*nx0*nky0*(3 + c),
 *   6 conventional flops per plane F = (3+2c)*T2D + 4M(1+c) + 3NxNy + 4M,
 *   with c = 1 if chi_has_v else 1/nv; 7: 1 if a fused (shared-memory resident) kernel is used, else 0;
 *   8: 1 if that kernel is the cluster kernel, 2 the group kernel, 4 its warp-autonomous form (gene_nl_set_plane_kernel), else 0.
 *   Returns NaN for an unknown `what` or NULL plan.
 */
double gene_nl_query(const gene_nl_plan* h, int what);

/*
 * gene_nl_compute_static -- rhs += scale * N(chi, g) WITHOUT A PLAN AND WITHOUT ANY ALLOCATION (the same
 * operation as gene_nl_compute with chi_has_v = 1: chi laid out like g, one chi plane per g plane).
 *
 * Why it exists.  gene_nl_create, gene_nl_set_* and the *_host entry points call cudaMalloc.  Some callers cannot:
 * a code that gives all device memory to its own pool at start-up (a later cudaMalloc fails), a time-step loop running
 * beside other streams (cudaMalloc / cudaFree synchronise the device and stall them), code inside a region where the
 * runtime forbids allocation.  This call allocates no device memory and no pinned host memory: no cudaMalloc, cudaFree,
 * cudaMallocHost, no stream or event creation.  The intermediate arrays of the planes in flight live in a
 * `static __device__` array inside the library (33.75 MiB + 5 KiB), which every GPU that loads the library holds until
 * the process exits, used or not.
 *
 * Limits (anything else returns GENE_NL_EUNSUPPORTED with a message that names the limit):
 *   nx0 = GENE_NL_STATIC_NX0 (96) and nky0 = GENE_NL_STATIC_NKY0 (48) exactly, i.e. the 144 x 144 padded grid of
 *   BASELINE.json configs[4]: the scratch is GENE_NL_STATIC_MAX_GROUPS (64) slots of 552 960 B, one per plane in flight,
 *   and a larger plane does not fit a slot;  nz*nv*nw*nspec <= GENE_NL_STATIC_MAX_PLANES.
 *   At most 64 SMs work (one plane each at a time): about 64/148 of the speed of gene_nl_compute on a B200.
 * Arguments: extents, kxmin, kymin as gene_nl_create; chi, g, rhs: DEVICE pointers, caller-owned, 16-byte aligned,
 * extents [nx0, nky0, nz, nv, nw, nspec], kx fastest (layout at the top of this file); rhs must not overlap chi or g.
 * `stream`: cudaStream_t as void* (NULL = legacy default stream).  Asynchronous: a counter clear and one kernel are
 * enqueued on `stream`; results equal gene_nl_compute's (same kernel code).  Errors as gene_nl_compute; on error before
 * the launch rhs is untouched.
 *
 * First call on each device: it looks up the device addresses of the static arrays (cudaGetSymbolAddress), copies the
 * root tables there with a synchronous cudaMemcpy and sets the kernel's shared-memory attribute, with that device
 * current.  Make that first call outside any stream capture; later calls do none of this.
 *
 * Sharing: every call on a device uses the same static array and finds the previous call's contents in it.  Nothing a
 * caller has to clear (the kernel overwrites each slot before reading it; the counters are cleared on `stream` by the
 * call itself).  But two calls that OVERLAP on the GPU -- different streams, or host threads on the same device -- write
 * the same slots and race: keep all calls on a device in one stream, or order them with events.  Plans
 * (gene_nl_compute*) have their own scratch and may run concurrently with it.
 */
#define GENE_NL_STATIC_NX0 96
#define GENE_NL_STATIC_NKY0 48
#define GENE_NL_STATIC_MAX_GROUPS 64
#define GENE_NL_STATIC_MAX_PLANES 2147483647LL
int gene_nl_compute_static(int nx0, int nky0, int nz, int nv, int nw, int nspec, double kxmin, double kymin,
                           const void* chi, const void* g, void* rhs, double scale, void* stream);

/* =====================================================================================================
 * x-GLOBAL VARIANT -- the operator the paper itself ran and timed (PAPER.md:39,
 * sect. 2.1-2.3): spectral in y only, real space in x.  PAPER.md:61: the fields are transposed, extended
 * in y by the 3/2 rule, transformed to real space, multiplied, transformed back, the additional modes are
 * deleted, the result is transposed, multiplied with a prefactor and added to the right-hand side.
 * "The nonlinear term needs as input four arrays, the x and y component of the ExB-velocity
 * and the derivatives of the distribution function with respect to x and y.  Additionally it needs the
 * already computed right-hand side".
 *
 *   per plane p and x:  N(x,y) = vex*dxg + vey*dyg  on the padded real grid Ny = 3*nky0,
 *                       rhs[x,j,p] += scale * pref[x] * N^(x,j),  j < nky0,  N^ = (1/Ny) sum_y N e^{-i ky y}
 *
 * Layout: every array (vex, vey, dxg, dyg, rhs) is complex128 [nx, nky0, planes], x fastest:
 * offset(x,j,p) = x + nx*(j + nky0*p); x is a real-space point, j the ky index (ky >= 0; ky < 0 implied by
 * reality; Im of the j = 0 entries is ignored).  pref: nx doubles (the x-dependent prefactor).
 * All pointers are DEVICE pointers, caller-owned, 16-byte aligned (pref: 8); rhs must not overlap an input.
 * Supported: nky0 in {8, 16, 32, 48, 64, 96, 128} (Ny = 24 .. 384); any nx >= 1 (tiles of 16 x points, 8 from
 * nky0 = 48 on; ragged tail allowed).
 * Asynchronous on `stream`; one kernel launch per compute.  Errors as for gene_nl_* (gene_nl_last_error).
 * gene_nlx_compute_host takes HOST pointers (same layouts; pref a host array of nx doubles) and streams the planes
 * through the device in chunks on three CUDA streams ("we split each input array into (usually four)
 * contiguous chunks of xy-planes, which are transferred and computed in two asynchronous CUDA streams"); 5 planes go
 * in and 1 comes out per plane computed.  SYNCHRONOUS; pinned host memory gives full overlap.
 * ===================================================================================================== */
typedef struct gene_nlx_plan gene_nlx_plan;

/* Returns NULL on failure (unsupported nky0, no device, out of memory). */
gene_nlx_plan* gene_nlx_create(int nx, int nky0, long long planes);

int gene_nlx_compute(gene_nlx_plan* h, const void* vex, const void* vey, const void* dxg, const void* dyg,
                     const double* pref, void* rhs, double scale, void* stream);

int gene_nlx_compute_host(gene_nlx_plan* h, const void* vex_host, const void* vey_host, const void* dxg_host,
                          const void* dyg_host, const double* pref_host, void* rhs_host, double scale);

/* NULL is a no-op.  Synchronises the device. */
void gene_nlx_destroy(gene_nlx_plan* h);

/* `what`: 0 planes, 1 Ny, 5 algorithmic bytes per plane (6 planes: 5 in, 1 out),
 * 6 conventional flops per plane (4 c2r + 1 r2c of length Ny per x at 2.5 N log2 N, multiply, prefactor+add). */
double gene_nlx_query(const gene_nlx_plan* h, int what);

#ifdef __cplusplus
}
#endif
#endif /* GENE_NL_H */
