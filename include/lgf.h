/* lgf.h -- C ABI of the B200-native Landau gauge fixer (steepest descent + Fourier acceleration).
 *
 * Method: arXiv 1208.1186 ("Landau gauge fixing using the steepest descent method
 * with Fourier acceleration"; GPU design PAPER.md:49-51).  PAPER.md prints none of the method's
 * formulas; the binding definition is the five steps of BASELINE.json `north_star`, restated in
 * SURVEY.md §8(a)/(c) and in DESIGN.md:
 *
 *   1. Delta(x) = sum_mu [U_mu(x-mu) - U_mu(x) - h.c.]_traceless,
 *      theta = (1/(3V)) sum_x Tr Delta Delta^+,   F = (1/(12V)) sum_x sum_mu Re Tr U_mu(x)
 *   2. 4D FFT of Delta's components
 *   3. scale mode k by p2max/p2(k), p2(k) = sum_mu 4 sin^2(pi k_mu/L_mu), zero mode dropped; inverse FFT
 *   4. g(x) = reunitarise(1 + (alpha/2) Delta~(x))     (row Gram-Schmidt, row 2 = conj(row0 x row1))
 *   5. U_mu(x) <- g(x) U_mu(x) g(x+mu)^+               (all sites from the old field)
 *
 * All compute runs in hand-written CUDA kernels for sm_100a on ONE GPU.  There is no CPU fallback:
 * every entry point that computes returns LGF_ECUDA if no CUDA device / kernel image is available.
 *
 * Conventions
 *   Sites are lexicographic with x fastest: s = x + Lx*(y + Ly*(z + Lz*t)), L = {Lx,Ly,Lz,Lt};
 *   mu = 0..3 <-> x,y,z,t; periodic in all four directions ("lexicographic layout").
 *   Link arrays AT THIS BOUNDARY are site-major AoS of full 3x3 matrices,
 *       links[s][mu][row][col][re,im]   (72 reals per site)
 *   with element type = the context precision (float for LGF_F32, double for LGF_F64), for BOTH
 *   storage modes.  LGF_REAL12 ("store only the first two rows (12 real numbers) and
 *   reconstruct the third row on the fly") drops row 2 on load and rebuilds it on store.
 *   A pointer argument is a HOST or a DEVICE pointer as stated by its `memspace` argument.
 *   Ownership: the caller owns every buffer it passes; the library copies in/out and keeps no
 *   reference after the call returns, except the workspace given to lgf_create, which must
 *   stay alive and untouched until lgf_destroy.
 *   Errors: 0 on success, a negative LGF_E* code otherwise; `*out` arguments are untouched on
 *   error.  No exceptions cross the ABI.  A context is not thread-safe.
 */
#ifndef LGF_H
#define LGF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lgf_ctx lgf_ctx; /* opaque, library-owned (host memory) */

enum { LGF_F32 = 0, LGF_F64 = 1 };         /* precision of links and of all per-site arithmetic   */
enum { LGF_REAL18 = 18, LGF_REAL12 = 12 }; /* reals stored per link on the device   */
enum { LGF_HOST = 0, LGF_DEVICE = 1 };     /* where a caller pointer lives                        */

enum {
    LGF_OK = 0,
    LGF_EINVAL = -1,       /* null pointer, L_mu < 2, bad enum, alpha <= 0, n < 0, workspace too small/misaligned */
    LGF_EUNSUPPORTED = -2, /* an L_mu with a prime factor other than 2 or 3, or a transform tile that
                              does not fit in shared memory (see lgf_workspace_bytes)               */
    LGF_ESTATE = -3,       /* iterate / fix / measure / store before load; any call but lgf_wait while an
                              lgf_iterate_async is pending */
    LGF_ECUDA = -4,        /* a CUDA call failed (no device, launch error, ...); see lgf_last_error */
    LGF_ENOMEM = -5        /* a host allocation failed */
};

/* Result of a measurement or of a run.  theta and F are those of the links held by the context when
 * the call returns (sums accumulated in fp64 in both precisions, fixed order: run-to-run identical). */
typedef struct {
    int64_t iterations; /* number of link updates applied by this call */
    double theta;       /* (1/(3V)) sum_x Tr Delta Delta^+   (north_star step 1) */
    double F;           /* (1/(12V)) sum_x sum_mu Re Tr U_mu(x) */
    int32_t converged;  /* theta < theta_tol (lgf_fix only; 0 otherwise) */
} lgf_result;

/* Bytes of device workspace lgf_create needs for this lattice: the links in the device layout, two packed
 * Delta-sized fields (4 complex per site: Delta / Delta~ and the layout-B spectrum between
 * K2 and K3), reduction partials, twiddle and p^2 tables, boundary staging.  About
 * (4 n_l + 16 (1 + 1/(2 Lz))) w bytes per site.  Returns 0 exactly when lgf_create would refuse the lattice:
 * invalid arguments, an extent that is not 2^a 3^b, V >= 2^31, or a transform tile that does not fit on chip. */
size_t lgf_workspace_bytes(const int32_t L[4], int precision, int storage);

/* Create a context.  `workspace_dev` is DEVICE memory of at least lgf_workspace_bytes(...) bytes,
 * 256-byte aligned, allocated and owned by the caller (e.g. a torch tensor); `cuda_stream` is a
 * cudaStream_t (NULL = the default stream) on which every kernel and copy of this context is
 * enqueued.  The library allocates only small host-side objects and one pinned host result block. */
int lgf_create(const int32_t L[4], int precision, int storage, void* workspace_dev,
               size_t workspace_bytes, void* cuda_stream, lgf_ctx** out);

/* north_star's three-argument form: allocates the workspace itself with cudaMalloc (freed by
 * lgf_destroy) and uses the default stream.  For C callers and tests. */
int lgf_create_simple(const int32_t L[4], int precision, int storage, lgf_ctx** out);

/* Batched context ("batching many small lattices per launch"): `nbatch` independent lattices of
 * the same shape, precision and storage are fixed by the SAME kernel launches (8^4 and 16^4 are launch-latency-bound
 * one at a time).  Every link array passed to lgf_load / lgf_store then holds the nbatch lattices back to
 * back (nbatch * V * 72 reals), and EVERY lgf_result pointer (lgf_measure, lgf_iterate, lgf_wait, lgf_fix,
 * lgf_profile_iterate) must point to an array of nbatch results, one per lattice.  Each lattice has its own theta, F,
 * iteration count and stopping test on the device: lgf_fix runs until every lattice has converged (or max_iter), and a
 * lattice's links stop changing at ITS crossing, so its result is the one a single-lattice context gives.
 * The inspection hooks and the Wilson-line calls are for single-lattice contexts (LGF_EUNSUPPORTED otherwise).
 * nbatch * ceil(Lz/2) * Lt must not exceed 65535.  lgf_create(...) == lgf_create_batch(..., 1, ...). */
size_t lgf_workspace_bytes_batch(const int32_t L[4], int precision, int storage, int32_t nbatch);
int lgf_create_batch(const int32_t L[4], int precision, int storage, int32_t nbatch, void* workspace_dev,
                     size_t workspace_bytes, void* cuda_stream, lgf_ctx** out);
int32_t lgf_batch_size(const lgf_ctx* ctx);

int lgf_destroy(lgf_ctx* ctx);

/* Copy a link field in (boundary layout above, element type = ctx precision).  Synchronous with
 * respect to the host: returns after the data has been consumed. */
int lgf_load(lgf_ctx* ctx, const void* links, int memspace);

/* Copy the current links out as full 3x3 matrices (row 2 rebuilt as conj(row0 x row1) in
 * LGF_REAL12 mode).  Synchronous. */
int lgf_store(lgf_ctx* ctx, void* links, int memspace);

/* Step 1 only: theta and F of the current links; out->iterations = 0. */
int lgf_measure(lgf_ctx* ctx, lgf_result* out);

/* Exactly n updates (steps 2-5, then step 1 on the new links), no stopping test.  n >= 0, alpha > 0.
 * One host synchronisation at the end.  (Which kernels run is the library's choice and lgf_describe reports it: most
 * lattices replay a five-kernel CUDA graph per update; an 8^4 lattice runs the whole call as ONE kernel on a 16-CTA
 * thread-block cluster that keeps the field in distributed shared memory.  Results agree to rounding.) */
int lgf_iterate(lgf_ctx* ctx, int64_t n, double alpha, lgf_result* out);

/* Same as lgf_iterate but only enqueues the work on the context's stream and returns; the result
 * is fetched (and the stream synchronised) by lgf_wait.  For device-side timing with CUDA events. */
int lgf_iterate_async(lgf_ctx* ctx, int64_t n, double alpha);
int lgf_wait(lgf_ctx* ctx, lgf_result* out);

/* Measure; while theta >= theta_tol and iterations < max_iter: update, measure (strict "<" test on
 * the updated links; SURVEY.md §8(c) reading #12).  The loop state lives on the device: iterations
 * after the crossing are skipped by a device-side flag, the host never synchronises per iteration.
 * Reaching max_iter is not an error (converged = 0). */
int lgf_fix(lgf_ctx* ctx, double alpha, double theta_tol, int64_t max_iter, lgf_result* out);

/* The step after the path (eq. (1): "e^{-F_singlet(r,T)/T + C} = (1/3) <Tr(W(r) W^+(0))>, where W(.) is the
 * temporal Wilson line"), evaluated on the links the context holds -- normally after lgf_fix, the quantity is not gauge
 * invariant.  For ONE configuration the average <.> is the average over the spatial lattice, Vs = Lx*Ly*Lz sites
 * xs = x + Lx*(y + Ly*z); the ensemble average and the fits of PAPER.md:78-80 are the caller's.
 *   lgf_wilson_lines:       lines[xs][row][col][re,im] = U_t(xs,0) U_t(xs,1) ... U_t(xs,Lt-1)   (9 Vs complex, ordered product)
 *   lgf_singlet_correlator: corr[r][re,im] = (1/(3 Vs)) sum_xs Tr[ W(xs + r) W(xs)^+ ], r = rx + Lx*(ry + Ly*rz), periodic
 *                           (Vs complex; corr[0] = 1, corr[-r] = conj corr[r])
 * Element type = ctx precision; host or device pointer per `memspace`; synchronous.  Both use the Delta fields as
 * scratch (the next lgf_iterate re-measures first); theta, F and the links are untouched. */
int lgf_wilson_lines(lgf_ctx* ctx, void* lines, int memspace);
int lgf_singlet_correlator(lgf_ctx* ctx, void* corr, int memspace);

/* Test/inspection hooks (device -> caller copies of intermediate fields of the LAST step executed):
 * the packed Delta field as [V][4] complex (c0 = D01, c1 = D02, c2 = D12, c3 = Im D00 + i Im D11),
 * element type = ctx precision.  After lgf_measure/lgf_iterate it holds Delta of the current links. */
int lgf_debug_get_delta(lgf_ctx* ctx, void* delta_packed, int memspace);
/* Runs steps 2-3 only on the current Delta field (in place) so that lgf_debug_get_delta returns
 * Delta~ (natural site order).  The links are untouched; call lgf_measure to restore Delta. */
int lgf_debug_fourier_accelerate(lgf_ctx* ctx);

/* Per-kernel timing of the iteration body: runs n updates like lgf_iterate but launches the five
 * kernels individually with CUDA events between them on the context's stream, and returns the
 * average device time in milliseconds of each: ms[0..4] = K2 fft_xy_fwd, K3 fft_zt_fwd_scale_inv,
 * K4 fft_xy_inv, K5 gbuild_update, K1 delta_theta_F.  For roofline reporting. */
int lgf_profile_iterate(lgf_ctx* ctx, int64_t n, double alpha, double ms[5], lgf_result* out);

/* Which kernels this context's iteration runs (for reports): info[0] = FFT path (0 runtime-radix,
 * 1 compile-time-sized one-tile-per-CTA, 2 pipelined persistent), info[1] = 1 if K5 and K1 are fused
 * into the marching update kernel (then ms[3] of lgf_profile_iterate is the fused kernel and ms[4] ~ 0),
 * info[2] = CTAs of the site kernel, info[3] = kernel launches per iteration (0 before the first run). */
int lgf_path_info(const lgf_ctx* ctx, int32_t info[4]);

/* Human-readable description of the kernels this context runs (which FFT path the lattice fell onto, line splits, tile
 * shapes, K5 flavour), NUL-terminated into buf[0..n): a lattice whose extents are not instantiated (e.g. a 32 x 16
 * (x,y) plane) runs on the slower one-tile-per-CTA or runtime-radix kernels, and this is where it says so. */
int lgf_describe(const lgf_ctx* ctx, char* buf, size_t n);

/* Number of kernel launches this context has enqueued since creation (for bench.py's gpu_launches). */
int64_t lgf_launch_count(const lgf_ctx* ctx);

/* Step 1 with NO allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): theta and F (north_star step 1; the definitions at the top of this file) of a link
 * field in the boundary layout above that already sits in DEVICE memory, with no context and no workspace.
 *   links_dev    device pointer, V*72 reals of `precision` (float / double), 16-byte aligned; read only
 *   cuda_stream  cudaStream_t (NULL = default stream); the two kernels are enqueued on it and the call returns WITHOUT
 *                synchronising (it records into a capturing stream like any launch)
 *   theta_F_dev  device pointer to 2 doubles, written by the second kernel: {theta, F}; sums in fp64, fixed order
 * Its only scratch, the per-CTA partial sums, is a static __device__ array of lgf_static_scratch_bytes() = 1 MiB that
 * EVERY GPU loading the library holds until the process exits; it bounds the lattice to LGF_STATIC_MAX_SITES sites
 * (64^4) -- larger lattices are refused with LGF_EINVAL and a message in lgf_static_last_error().  All calls share the
 * array: calls whose kernels may overlap on the GPU (different streams, parallel graph branches) race on it; calls on
 * one stream are safe.  Nothing in it needs clearing between calls.  The call uses no cudaMalloc, cudaFree or
 * allocating library routine.  lgf_static_init() resolves the array's device address for the CURRENT device (once per
 * device; lgf_measure_static does it itself on first use, so calling it is only needed to keep that first-use work out
 * of a capture or a timed loop).  Errors: LGF_EINVAL (null pointer, bad precision, L_mu < 2, too many sites),
 * LGF_ECUDA (symbol lookup or launch failed). */
#define LGF_STATIC_MAX_SITES 16777216
int lgf_static_init(void);
int lgf_measure_static(const int32_t L[4], int precision, const void* links_dev, void* cuda_stream, double* theta_F_dev);
size_t lgf_static_scratch_bytes(void);
/* Text of the last error of this thread's lgf_static_* / lgf_measure_static calls ("" if none). */
const char* lgf_static_last_error(void);

const char* lgf_strerror(int code);
/* Text of the last CUDA error seen by this thread's calls ("" if none). */
const char* lgf_last_error(void);
/* "x.y" version string. */
const char* lgf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LGF_H */
