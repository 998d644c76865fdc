/*
 * sc.h -- C ABI of libsc: real-space convolution of a HEALPix map (RING ordered; NESTED is reordered on
 * the device) with a compact, radially symmetric kernel on one NVIDIA B200 (sm_100a).
 *
 * The operation (BASELINE.json north_star; the "real-space portion" that the paper runs on the
 * GPU -- PAPER.md:66 section 2, Fig. 1 caption -- i.e. "convolving a ... map with a
 * radial kernel", with the real-space kernel truncated at theta_cut):
 *
 *     out_b(p) = Omega_pix * SUM_{q : theta_pq <= theta_max} K(cos theta_pq) * m_b(q),
 *     Omega_pix = 4 pi / N_pix,  N_pix = 12 nside^2,  b = 0 .. B-1 (maps sharing one kernel).
 *
 * Inclusion (reading R4) is decided exactly as the fp64 test
 *     z_p z_q + (s_p s_q) cos(phi_p - phi_q) >= cos(theta_max)
 * evaluated in IEEE double without FMA contraction (the self pair is included); K is the linear
 * interpolant of the caller's table in cos(theta) (PAPER.md:106 speaks of interpolating the
 * real-space kernel from nodes; node placement here is uniform in cos theta, reading R5, or the paper's
 * two-zone placement through sc_plan_create_zoned, reading R11);
 * products and sums are fp32 on the device ("single-precision arithmetic in the GPU",
 * PAPER.md:124).
 *
 * Conventions
 *   - Nothing throws or aborts across this boundary: every entry point returns an sc_status and
 *     leaves its outputs untouched on failure.
 *   - "HOST" / "DEVICE" below say where a pointer must live.  The library never allocates or
 *     frees memory the caller passes in; a plan owns its own device tables.
 *   - A plan belongs to the CUDA device that was current when it was created and is immutable
 *     afterwards; it may be used from one stream at a time.
 *   - There is no CPU fallback: without a usable CUDA device sc_plan_create returns SC_ERR_CUDA.
 */
#ifndef SC_H
#define SC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct sc_plan sc_plan; /* opaque */

typedef enum {
    SC_OK = 0,
    SC_ERR_INVALID_ARG = 1, /* NULL where not allowed, nside < 1, n_table < 2, theta_max out of range, B < 1 ... */
    SC_ERR_UNSUPPORTED = 2, /* 12 nside^2 >= 2^31; knife-edge list overflow; latitude bands on a NESTED plan */
    SC_ERR_ALLOC = 3,       /* host or device allocation failed */
    SC_ERR_CUDA = 4         /* no device / a CUDA call failed (sc_last_cuda_error() names it) */
} sc_status;

enum { SC_ORDER_RING = 0, SC_ORDER_NESTED = 1 };   /* NESTED: nside must be a power of two */

/* Which kernels sc_convolve may use (debug / measurement knob; results are the same operation). */
enum {
    SC_PATH_AUTO = 0,     /* fastest available for every ring (default) */
    SC_PATH_GENERIC = 1   /* one thread per output pixel everywhere (the simple reference kernel) */
};

/*
 * sc_plan_create -- precompute everything that depends only on (nside, kernel, theta_max).
 *   plan       HOST  out: receives the new plan (unchanged on failure).
 *   nside      HEALPix resolution, >= 1, need not be a power of two; 12 nside^2 < 2^31.
 *   ordering   SC_ORDER_RING, or SC_ORDER_NESTED (nside a power of two): maps passed to sc_convolve /
 *              sc_convolve_host are then NESTED ordered; the plan owns RING work buffers (2 x min(max_batch, 4)
 *              maps) and reorders on the device around the same kernels.  Latitude bands need RING.
 *   ktable     HOST  n_table doubles, K sampled at x_i = c + i (1 - c)/(n_table - 1),
 *              c = cos(theta_max), i.e. ktable[0] = K(cos theta_max), ktable[n_table-1] = K(1).
 *              Copied; the caller may free it after the call.
 *   n_table    >= 2.
 *   theta_max  radians, 0 < theta_max <= pi/2.
 *   max_batch  >= 1: largest B later passed to sc_convolve (larger B still works, in chunks).
 * Work done: ring geometry tables (fp64 and fp32), the device interpolation table, per-ring
 * input-ring intervals, and one audit pass on the GPU that counts all pairs and collects
 * "knife-edge" pairs (|dot - c| below a few ulp) whose inclusion is then decided on the host
 * with the host libm (DESIGN.md section "Bit-exact inclusion").  Synchronous.
 */
sc_status sc_plan_create(sc_plan **plan, int nside, int ordering, const double *ktable,
                         int n_table, double theta_max, int max_batch);

/*
 * sc_plan_create_zoned -- the same with the paper-style two-zone table ("we place half the
 * available interpolation nodes within the first 1/16 of the available support"; reading R11).
 *   n_table    even, >= 4; h = n_table / 2.
 *   zone_frac  0 < zone_frac < 1 (the paper: 1/16); x1 = cos(zone_frac * theta_max).  0 = uniform table.
 *   ktable     K at the nodes  x_i = c + i (x1 - c) / h            for i <  h  (outer zone),
 *                              x_i = x1 + (i - h)(1 - x1) / (h - 1) for i >= h  (inner zone, next to theta = 0),
 *              linear interpolation in x = cos(theta) between adjacent nodes.
 * The inner zone must be at least as dense as the outer one ((h - 1)/(1 - x1) >= h/(x1 - c)), otherwise
 * SC_ERR_INVALID_ARG.  Everything else as sc_plan_create.
 */
sc_status sc_plan_create_zoned(sc_plan **plan, int nside, int ordering, const double *ktable,
                               int n_table, double theta_max, double zone_frac, int max_batch);

/*
 * sc_convolve -- the hot path.  Enqueues the convolution of B maps on `cuda_stream` and returns
 * without synchronising the host.
 *   in_maps    HOST array of B DEVICE pointers, each to N_pix fp32 values (RING order),
 *              16-byte aligned.
 *   out_maps   HOST array of B DEVICE pointers, each to N_pix fp32 values, 16-byte aligned;
 *              must not overlap any input or any other output (SC_ERR_INVALID_ARG).  Fully overwritten.
 *   B          >= 1.
 *   cuda_stream  a cudaStream_t (CUstream) passed as void*; NULL = the legacy default stream.
 * Map values are plain numbers: no bad-pixel sentinel is interpreted (paper silent).
 * Only kernel launches are enqueued (no allocation, no host synchronisation), so the call may be
 * captured into a CUDA graph.  The plan itself is not modified apart from the launch counter read by
 * sc_last_launch_count; a NESTED plan routes the maps through its plan-owned RING work buffers (sized at plan
 * creation for min(max_batch, 4) maps; larger batches run in chunks of that size), so -- like every plan -- it
 * serves one stream at a time.
 */
sc_status sc_convolve(const sc_plan *plan, const float *const *in_maps, float *const *out_maps,
                      int B, void *cuda_stream);

/*
 * sc_convolve_host -- the same operation with HOST buffers (the end-to-end call): copies the B
 * input maps to plan-owned device staging buffers, runs the kernels of sc_convolve, copies the results
 * back and synchronises.  On the AUTO path the three steps are pipelined over latitude chunks on three
 * streams (a chunk is computed as soon as its rows have arrived and returned while later chunks are
 * still in flight); the results are identical to sc_convolve's.  in/out: HOST arrays of B HOST pointers to N_pix fp32 each (pinned memory makes
 * the copies faster but is not required).
 */
sc_status sc_convolve_host(sc_plan *plan, const float *const *in_maps_host,
                           float *const *out_maps_host, int B);

/* Destroy a plan and free its device memory.  NULL is allowed. */
sc_status sc_plan_destroy(sc_plan *plan);

/* Select the kernel path used by later sc_convolve calls on this plan (SC_PATH_*). */
sc_status sc_plan_set_path(sc_plan *plan, int path);

/*
 * sc_plan_info -- facts about a plan.  Any output pointer may be NULL.
 *   npix            12 nside^2
 *   total_pairs     number of included (p, q) pairs over the whole sphere, self pairs included
 *                   (from the audit pass)
 *   cos_theta_max   the threshold c used by the inclusion test
 *   n_knife_edge    number of pairs that were decided on the host
 */
sc_status sc_plan_info(const sc_plan *plan, int64_t *npix, int64_t *total_pairs,
                       double *cos_theta_max, int64_t *n_knife_edge);

/*
 * sc_debug_neighbour_counts -- verification only, not part of the timed path.  For every pixel
 * p writes the number of included neighbours to count_dev[p] and, if sig_dev != NULL, the sum of
 * the neighbours' RING indices to sig_dev[p].  Both DEVICE pointers, N_pix entries (entry p refers to pixel p
 * in the plan's ordering; the signature sums RING indices also for NESTED plans; NESTED: synchronous).
 * Runs the one-thread-per-pixel generic kernel in count mode, i.e. the inclusion code of SC_PATH_GENERIC (fp32
 * table coordinate with a guard band, canonical fp64 test inside it).  sym_kernel and belt_kernel decide
 * inclusion with their own fp32 form and the same fp64 test inside their guard band; THEIR sets are verified
 * through the convolution itself (K == 1 table, small-integer maps: tests/test_gpu_parity.py
 * test_exact_integer_sums_fast_kernels).  Asynchronous on cuda_stream.
 */
sc_status sc_debug_neighbour_counts(const sc_plan *plan, int32_t *count_dev, uint64_t *sig_dev,
                                    void *cuda_stream);

/*
 * sc_neighbour_counts_static -- sc_debug_neighbour_counts for callers that must not allocate (CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): same arguments, same results, asynchronous on cuda_stream for
 * RING and NESTED plans alike, and no cudaMalloc / cudaFree or other allocating call.  The RING-ordered scratch that
 * a NESTED plan needs (4 + 8 bytes per pixel) lives in a static device array of SC_STATIC_MAX_NPIX entries (2.25 MiB
 * that every GPU loading the library holds until exit), so 12 nside^2 <= SC_STATIC_MAX_NPIX, i.e. nside <= 128
 * (larger: SC_ERR_UNSUPPORTED, nothing launched).  The plan's device must be current on a device's first call
 * (SC_ERR_INVALID_ARG otherwise): that call resolves the array's device address (cudaGetSymbolAddress), so make it
 * outside stream capture.  All calls on a device share the array, which keeps the previous call's contents (every
 * entry used is overwritten before it is read: nothing needs clearing); calls that OVERLAP on the GPU -- different
 * streams, concurrent graph replays -- race on it and must be serialised by the caller.
 */
#define SC_STATIC_MAX_NPIX 196608
sc_status sc_neighbour_counts_static(const sc_plan *plan, int32_t *count_dev, uint64_t *sig_dev, void *cuda_stream);

/*
 * sc_debug_stats -- numbers gathered by the audit pass at plan creation (HOST outputs, may be NULL):
 *   n_uncertain   pairs whose fp32 table coordinate fell inside the guard band and were therefore
 *                 re-decided in fp64 on the device
 *   max_t_err     max |t_fp32 - t_fp64| (table cells) seen over those pairs
 *   guard_band    half-width of the guard band (table cells)
 */
sc_status sc_debug_stats(const sc_plan *plan, int64_t *n_uncertain, double *max_t_err,
                         double *guard_band);

/*
 * sc_convolve_profile -- measurement only: the same launches as sc_convolve with CUDA events recorded
 * on `cuda_stream` around every kernel; synchronises the stream and returns the device time of each
 * kernel of the step, summed over batch chunks:
 *   ms[SC_K_POLAR]  generic_warp_kernel  (rings next to the poles)
 *   ms[SC_K_SYM]    sym_kernel           (polar caps and the cap/belt transition)
 *   ms[SC_K_BELT]   belt_kernel          (equatorial belt stencil)
 * ms: HOST array of SC_K_COUNT floats (milliseconds; 0 for a kernel this plan does not launch).
 */
enum { SC_K_POLAR = 0, SC_K_SYM = 1, SC_K_BELT = 2, SC_K_COUNT = 3 };
sc_status sc_convolve_profile(const sc_plan *plan, const float *const *in_maps,
                              float *const *out_maps, int B, void *cuda_stream, float *ms);

/*
 * sc_plan_partition -- which pixels each kernel of the AUTO path writes (HOST outputs, may be NULL).
 * With N = nside, base rings are 1 .. 2N and every base ring r stands for itself and its southern
 * mirror 4N - r:
 *   polar_rings      base rings 1 .. polar_rings                     -> generic_warp_kernel
 *   first_belt_ring  base rings polar_rings + 1 .. first_belt_ring-1 -> sym_kernel,
 *                    base rings first_belt_ring .. 2N                 -> belt_kernel
 *                    (2N + 1 if the plan has no belt kernel; polar_rings = 2N if it has no fast path)
 */
sc_status sc_plan_partition(const sc_plan *plan, int *polar_rings, int *first_belt_ring);

/*
 * Latitude bands ("the sky map [can] be divided into latitude bands with minimal overlap ...
 * convolution on the latitude bands is completely independent once the necessary overlap is included").
 * A band is a range of BASE rings lo .. hi (1 <= lo <= hi <= 2 nside) together with the southern mirror
 * rings 4 nside - hi .. 4 nside - lo, because the kernels evaluate a pair geometry once for both.
 *
 * sc_band_partition -- band `rank` of a split of the sphere into `world` bands of nearly equal estimated
 * work (cap pixels cost more than belt pixels; 1 <= world <= 2 nside).  HOST outputs, any may be NULL:
 *   ring_lo, ring_hi   the band's base rings
 *   out_rows[4]        pixel ranges [o0, o1) U [o2, o3) the band's convolution writes
 *   in_rows[4]         pixel ranges [i0, i1) U [i2, i3) it reads (band + theta_max overlap); a range may be
 *                      empty (x2 == x3) when the two parts merge at the equator
 *
 * sc_convolve_band -- sc_convolve restricted to one band: reads only in_rows of every input map, writes
 * only out_rows of every output map (the other pixels are not touched).  Maps are full-size N_pix
 * buffers as in sc_convolve, so rows exchanged between ranks land at their global positions.  The first
 * call for a new band builds its tile list (synchronous); later calls are asynchronous on the stream.
 */
sc_status sc_band_partition(const sc_plan *plan, int world, int rank, int *ring_lo, int *ring_hi,
                            int64_t *out_rows, int64_t *in_rows);
sc_status sc_convolve_band(sc_plan *plan, int ring_lo, int ring_hi, const float *const *in_maps,
                           float *const *out_maps, int B, void *cuda_stream);

/*
 * North polar cap only ("orienting the ... maps such that the survey area lies in the polar cap, reducing
 * the number of rings"): a partial-sky map rotated so that the survey covers rings 1 .. ring_hi of the northern
 * hemisphere.  sc_convolve_cap computes exactly those output rings; unlike a latitude band it evaluates NO southern
 * mirror images (north-only kernel instance: 4 rotations x the reflection phi -> pi/2 - phi share a pair geometry) and
 * reads nothing beyond the disc of ring ring_hi, so the map buffers need only hold the rows given by sc_cap_rows.
 *
 * sc_cap_rows -- HOST outputs (may be NULL): out_rows[2] = pixel range [0, o1) written (rings 1 .. ring_hi),
 *   in_rows[2] = pixel range [0, i1) read (rings up to ring_hi + theta_max overlap).  1 <= ring_hi <= 2 nside.
 * sc_convolve_cap -- in_maps / out_maps: HOST arrays of B DEVICE pointers to at least in_rows[1] / out_rows[1] fp32
 *   values (RING order from the north pole), 16-byte aligned, not overlapping.  Pixels >= out_rows[1] are not touched.
 *   Maps are processed one per launch.  RING plans only (SC_ERR_UNSUPPORTED for NESTED).  The first call for a new
 *   ring_hi builds its tile list (synchronous); later calls are asynchronous on the stream.
 */
sc_status sc_cap_rows(const sc_plan *plan, int ring_hi, int64_t *out_rows, int64_t *in_rows);
sc_status sc_convolve_cap(sc_plan *plan, int ring_hi, const float *const *in_maps, float *const *out_maps, int B,
                          void *cuda_stream);

/*
 * sc_debug_fma_peak -- measurement only: the sustained FP32 FMA rate of the current device, measured with a
 * register-only loop of independent FMA chains (packed = 0: scalar FFMA; packed = 1: FFMA2, the packed form the
 * convolution kernels accumulate with) on 2 x 1024 threads per SM, best of 3 launches of a few ms.  bench.py uses
 * it as the measured denominator of the roofline.  packed = 2: FFMA2 with the operand pattern of the
 * kernels' accumulation (accumulator pair += tap pair x map value, 16 warps per SM): what the register file sustains
 * for that pattern, reported next to the peak.  Other values: SC_ERR_INVALID_ARG.
 *   fma_per_s   HOST out: fp32 fused multiply-adds per second (an FFMA2 counts as two)
 *   elapsed_ms  HOST out (may be NULL): duration of the best launch
 * Synchronous on the legacy default stream; needs no plan.
 */
sc_status sc_debug_fma_peak(int packed, double *fma_per_s, double *elapsed_ms);

/* Kernel launches enqueued by the last sc_convolve / sc_convolve_host on this plan. */
int sc_last_launch_count(const sc_plan *plan);

/*
 * sc_plan_double_coordinate -- 1 if the plan's kernels form the table coordinate t = (1 - cos theta_pq) (n-1)/(1-c) of every
 * pair in fp64 (and split it into table cell + position in the cell), 0 if in fp32.  Chosen at plan creation from the
 * table alone: fp32 resolves t to ~t 2^-23 cells, i.e. K to |slope of cell j| j 2^-23; if that, rms over the cells,
 * exceeds 6.5e-7 of the table's rms -- oscillating tables such as the real-space part of the paper's least-squares
 * split (Fig. 4) at theta_cut of degrees -- fp32 geometry alone would break the 1e-6 bar (DESIGN.md
 * section 10; the paper reports this single-precision sensitivity as alpha = 5).  Such plans run one map
 * per launch through the 16-image sym instance, the belt stencil (taps in fp64) and the generic kernels; the two-zone
 * table is not combined with it.  Products and sums stay fp32.  NULL plan: 0.
 */
int sc_plan_double_coordinate(const sc_plan *plan);

const char *sc_status_string(sc_status s);
/* Text of the last CUDA error seen by this library on the calling thread ("" if none). */
const char *sc_last_cuda_error(void);
/* Library version, e.g. "sc 0.2 (sm_100a)". */
const char *sc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SC_H */
