/*
 * corr.h -- C ABI of libcorr.so: the X-engine of an FX software correlator on NVIDIA B200 (sm_100a).
 *
 * What it computes (Wang & Harris, arXiv:1305.5639; Sec. 2, Eq. 2):
 *
 *     V_ij[c] = sum_{t=0}^{T-1} conj(x_i[t][c]) * x_j[t][c]
 *
 * for every frequency channel c, every station pair i >= j INCLUDING the autocorrelations i == j
 * ("triangle pattern for all non-redundant pairs", Sec. 4; autocorrelations on the
 * hypotenuse, Sec. 4.2) and all P x P polarisation products, as raw sums (Eq. 2 has
 * no normalisation), optionally integrated across successive calls ("results are usually then
 * accumulated", Sec. 2).
 *
 * Every function is extern "C", never throws and never aborts the process.  Pointers are plain; each
 * argument says whether it is a HOST or a DEVICE pointer.  The library links only the CUDA
 * runtime; callers may use anything (e.g. PyTorch) for device memory and streams.
 * Device-side watchdog: the tensor-core kernels wait on hardware barriers; should one not complete
 * within 2^33 SM clocks (seconds; a legitimate wait is microseconds) the kernel traps instead of
 * hanging the GPU, the stream reports a launch failure (CORR_ECUDA from the next call that checks)
 * and the CUDA context is unusable afterwards, as after any device-side fault.
 * Devices: compute capability 10.0 only (B200 / GB200); the library carries sm_100a code, no PTX.
 *
 * Layouts (C-contiguous, fastest axis last)
 *   in   [n_time][n_chan][n_station][n_pol] complex, (re, im) interleaved:
 *          CORR_CI8  : 2 x int8  per sample (2 bytes);  any value in [-128, 127] is exact
 *          CORR_CF16 : 2 x IEEE binary16 per sample (4 bytes); values must be finite
 *   out  [n_chan][B][n_pol][n_pol] complex, (re, im) interleaved, B = n_station(n_station+1)/2:
 *          CORR_CI8  : 2 x int32 (8 bytes per visibility), exact
 *          CORR_CF16 : 2 x fp32  (8 bytes per visibility), fp32 accumulation
 *        baseline b(i,j) = i(i+1)/2 + j for j <= i (corr_baseline_index); the first polarisation
 *        axis p belongs to the conjugated station i, the second (q) to station j.  Autocorrelation
 *        rows keep all P x P products, so V_ii^{XY} and V_ii^{YX} = conj(V_ii^{XY}) are both stored.
 *
 * Threading: one handle is used from one host thread at a time; handles are independent.
 */
#ifndef CORR_H_
#define CORR_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct corr_plan* corr_handle;

/* dtype */
enum { CORR_CI8 = 0, CORR_CF16 = 1 };

/* return codes */
enum {
    CORR_OK = 0,
    CORR_EINVAL = -1,        /* bad argument (size, NULL pointer, alignment, unknown enum)       */
    CORR_EUNSUPPORTED = -2,  /* no CUDA device, or the device is not compute capability 10.x     */
    CORR_ENOMEM = -3,        /* host or device allocation failed                                 */
    CORR_ECUDA = -4,         /* a CUDA call failed; corr_last_error() carries the CUDA string    */
    CORR_EOVERFLOW = -5      /* CORR_CI8: integration would exceed the exact int32 range         */
};

/* which kernel corr_xengine launches (corr_set_kernel); all compute the same result */
enum {
    CORR_KERNEL_AUTO = 0,    /* default: chosen from the geometry (see corr_get_kernel)                              */
    CORR_KERNEL_SINGLE = 1,  /* tcgen05, one CTA per 128 x 256 tile of the per-channel Gram matrix                   */
    CORR_KERNEL_PAIR = 2,    /* tcgen05 cta_group::2: a CTA pair per 256 x 256 tile (half the L2 bytes per MAC of B)  */
    CORR_KERNEL_SIMT = 3     /* CUDA-core kernel for geometries TMA cannot address (and a cross-check)                */
};

/*
 * corr_create -- plan for one problem geometry on the CURRENT CUDA device (host call).
 *   n_station >= 1, n_pol in {1, 2}, n_chan >= 1, n_time >= 1, dtype in {CORR_CI8, CORR_CF16}.
 * Builds the triangular tile schedule (only tiles touching s_i >= s_j are scheduled), uploads it,
 * and sizes the workspace.  Returns NULL on failure; the reason is corr_last_error(NULL).
 * The handle owns its device allocations until corr_destroy.
 */
corr_handle corr_create(int n_station, int n_pol, int n_chan, int n_time, int dtype);

/*
 * corr_create_window -- plan for a CHANNEL WINDOW of a larger problem.  Eq. 2 is independent per
 * frequency channel (the paper's "orthogonal correlation triangles separating frequency channels prior to the CMAC
 * stage"), so several handles -- on one GPU or one per GPU / process -- can each integrate a block of
 * channels of ONE input into their own slabs of ONE output with no communication.  The handle processes channels
 * [chan0, chan0 + n_chan) of buffers laid out for n_chan_total channels, IN PLACE:
 *   in   [n_time][n_chan_total][n_station][n_pol]  -- the whole-band buffer; only the window's columns are read
 *   out  [n_chan_total][B][n_pol][n_pol]           -- the whole-band buffer; only slabs chan0 .. chan0 + n_chan - 1 are
 *                                                     written (or accumulated into); every other byte is left untouched
 * corr_input_bytes / corr_output_bytes report the WHOLE-BAND sizes.  0 <= chan0, 1 <= n_chan, chan0 + n_chan <=
 * n_chan_total.  Everything else (corr_xengine, corr_xengine_dumps, corr_xengine_host, accumulate, errors) as for
 * corr_create; corr_create(N, P, C, T, d) == corr_create_window(N, P, C, 0, C, T, d).  corr_corner_turn is not
 * available on a window plan.  With corr_xengine_host only the window's input columns and output slabs cross the bus.
 */
corr_handle corr_create_window(int n_station, int n_pol, int n_chan_total, int chan0, int n_chan, int n_time, int dtype);

/*
 * corr_xengine -- one integration of n_time samples (Eq. 2), asynchronous on `stream`.
 *   in         DEVICE pointer, corr_input_bytes(h) bytes, 16-byte aligned, layout above; must stay
 *              valid and unmodified until `stream` has passed this call.  Not written.
 *   out        DEVICE pointer, corr_output_bytes(h) bytes, 16-byte aligned, layout above.
 *              accumulate == 0: every word is overwritten (no pre-zeroing needed).
 *              accumulate != 0: out <- out + V; `out` must hold an earlier result of the same geometry.
 *   stream     a cudaStream_t passed as void* (NULL = the legacy default stream).
 * Returns CORR_OK or a negative code.  CORR_CI8 with accumulate != 0 returns CORR_EOVERFLOW,
 * launching nothing, once the samples integrated through this handle since the last accumulate == 0
 * call would exceed 65535 (|V| <= 2 * 128^2 * T_total must fit int32).
 * CUDA graphs: everything the call does on the device is enqueued on `stream` (one kernel; on the pair kernel a 4-byte
 * memset of its tile-feed counter in front), so a sequence of calls can be captured with stream capture and replayed --
 * the way to run launch-bound geometries (config 1: 13 us per call eagerly, 4.8 us replayed).  Call once before
 * capturing (the first call on a handle encodes its tensor map on the host); the overflow accounting above is done at
 * CAPTURE time, replays do not advance it.  A captured pair-kernel launch has ONE of the handle's 256 tile-feed counters
 * (and the memset that clears it) baked into the graph, while later launches on the handle keep walking the ring: once
 * calls of this handle have been captured, do not run that graph concurrently with other launches of the SAME handle on
 * another stream (after 256 further launches they would share the counter and tiles would be skipped or done twice).
 * Replays and eager calls ordered on one stream, or concurrent work on DIFFERENT handles, are fine.
 */
int corr_xengine(corr_handle h, const void* in, void* out, int accumulate, void* stream);

/*
 * corr_xengine_host -- same operation with HOST buffers (blocking; layouts and sizes as corr_xengine).  The plan's
 * channels are cut into up to 8 windows that flow through a three-stage pipeline on the handle's own streams: the
 * host-to-device copy of window w+1 (a strided 2-D copy straight out of `in_host`), the X-engine kernel on window w,
 * and the device-to-host copy of window w-1's output slab overlap, so the bus runs in both directions while the GPU
 * computes.  The handle owns the device staging (two input windows + the running output).  With accumulate != 0 the
 * running sum lives in that device buffer (state of the previous corr_xengine_host call on this handle) and
 * `out_host` receives the updated integration; `out_host` may be NULL to leave the running sum on the device until a
 * later call asks for it.  Returns after all copies have completed.  PINNED host memory is needed for the copies to
 * overlap (pageable memory works but serialises).  CORR_EOVERFLOW as corr_xengine.
 * On failure: the call returns only after everything it had queued has drained, so `in_host` / `out_host` may be freed
 * or reused at once; the running sum on the device is then incomplete and is marked invalid -- the next call must start a
 * new integration (accumulate == 0; accumulate != 0 returns CORR_EINVAL), and the contents of `out_host` are undefined.
 */
int corr_xengine_host(corr_handle h, const void* in_host, void* out_host, int accumulate);

/*
 * Rectangular, cross-only X-engine.  PAPER.md:79, Sec. 4: in the space-division models "some
 * of the nodes ... need to process two parts of the input streams in a rectangle pattern for cross-correlations
 * only".  For two station groups A (n_station_a) and B (n_station_b) sharing n_pol, n_chan, n_time and dtype:
 *
 *     out[c][i][j][p][q] = sum_t conj(in_a[t][c][i][p]) * in_b[t][c][j][q]        (Eq. 2, i in A, j in B)
 *
 * every (i, j) is stored: no triangle, no autocorrelations.  Layouts as for corr_xengine with
 *   in_a [n_time][n_chan][n_station_a][n_pol], in_b [n_time][n_chan][n_station_b][n_pol]   (DEVICE, 16-byte aligned)
 *   out  [n_chan][n_station_a][n_station_b][n_pol][n_pol] complex int32 / fp32               (DEVICE, 16-byte aligned)
 * corr_input_bytes(h) is the size of in_a, corr_input_bytes_b(h) of in_b, corr_output_bytes(h) of out.
 * corr_create_cross returns NULL on failure (corr_last_error(NULL)); the handle is used with corr_xengine_cross
 * only (corr_xengine, corr_xengine_host and corr_corner_turn return CORR_EINVAL on it, and corr_xengine_cross
 * returns CORR_EINVAL on a corr_create handle).  accumulate / stream / CORR_EOVERFLOW exactly as corr_xengine.
 * Runs on the CTA-pair tcgen05 kernel (full rectangle of 256 x 256 tiles, group A and group B read in place through
 * two tensor maps) or, when a group's per-channel row is not a multiple of 16 bytes, on the SIMT kernel.
 */
corr_handle corr_create_cross(int n_station_a, int n_station_b, int n_pol, int n_chan, int n_time, int dtype);
int corr_xengine_cross(corr_handle h, const void* in_a, const void* in_b, void* out, int accumulate, void* stream);
size_t corr_input_bytes_b(corr_handle h);    /* cross plans: T*C*Nb*P * (2 or 4); else 0 */

/*
 * corr_xengine_dumps -- short-integration mode (the paper's "transient detector ... between
 * conjugate multiplications and accumulations" wants visibilities every few samples): the n_time samples
 * of `in` are cut into n_dump consecutive integrations of n_time / n_dump samples, each integrated SEPARATELY (Eq. 2
 * per integration, no sum across them) in ONE kernel launch.
 *   in     DEVICE, as for corr_xengine ([n_time][n_chan][n_station][n_pol]; integration d = samples
 *          [d * n_time/n_dump, (d+1) * n_time/n_dump)).
 *   out    DEVICE, n_dump * corr_output_bytes(h) bytes: [n_dump][n_chan][B][n_pol][n_pol] complex int32 / fp32;
 *          every word is overwritten (there is no accumulate).
 *   n_dump must divide n_time.  HERK plans only (CORR_EINVAL on a cross plan).  Runs on the CTA-pair kernel for every
 *   TMA-addressable geometry (rank-3 tensor map: a TMA box never crosses into the next integration), else SIMT.
 */
int corr_xengine_dumps(corr_handle h, const void* in, void* out, int n_dump, void* stream);

/*
 * corr_fengine -- the F-engine in front of the X-engine.  PAPER.md:49-52 (Sec. 2, Eq. 1):
 *     S[k] = sum_{n=0}^{N-1} s[n] exp(-j (2 pi / N) k n),   N = 256 ("An FFT length of 256 is used across all tests",
 * PAPER.md:176), applied to consecutive non-overlapping blocks of each stream's 8-bit REAL samples.
 *   in    DEVICE, 16-byte aligned: int8 [n_stream][n_spectra * 256], each stream contiguous in time.
 *   out   DEVICE, 4-byte aligned: complex fp16 (re, im) [n_spectra][128][n_stream]: the 128 non-redundant channels
 *         k = 0..127 of every block (real input: S[256 - k] = conj(S[k]); the Nyquist bin is dropped), raw sums
 *         (|S| <= 128 * 256 fits fp16), computed in fp32 and rounded to nearest.  With n_stream = n_station * n_pol
 *         (stream m = s * n_pol + p) this IS corr_xengine's CORR_CF16 input [n_time = n_spectra][n_chan = 128]
 *         [n_station][n_pol]: no corner turn between the engines.
 * Stateless (no handle), asynchronous on `stream`; CORR_OK or a negative code, message via corr_last_error(NULL).
 * Kernels: with n_stream a multiple of 8 and at least 32 (whole half tiles of 64 streams plus at most one ragged one whose
 * padding does not more than double the work: 32, 40, ..., 64, 72, 96, 200, ...) and a 16-byte aligned `out` the transform
 * runs as a dense contraction on the
 * tcgen05 tensor cores (the real-input DFT folded onto 128 samples, twiddle matrices split into fp16 hi + lo parts,
 * fp32 accumulation: csrc/fengine_tc.cuh); every other geometry runs on the CUDA-core radix-16 x 16 FFT kernel
 * (csrc/fengine.cuh).  Both meet the same bound against the fp64 definition: 0.5 ulp of the fp16 output plus
 * 2e-6 sum_n |s[n]|.  corr_fengine_simt forces the CUDA-core kernel (cross-check); corr_fengine_uses_tensor_cores tells
 * which one corr_fengine would launch on the CURRENT device (1 / 0): it applies the same two tests as corr_fengine itself,
 * the geometry / alignment rule above and the per-device set-up of the tensor-core kernel (0 on a device that is not
 * sm_100, or where that set-up failed; calling it may perform the set-up, which allocates the 160 KB twiddle table).
 */
int corr_fengine(const void* in, void* out, int n_stream, long long n_spectra, void* stream);
int corr_fengine_simt(const void* in, void* out, int n_stream, long long n_spectra, void* stream);
int corr_fengine_uses_tensor_cores(int n_stream, const void* out);

/*
 * corr_fengine_ci8 -- the same transform with REQUANTISED complex int8 output, the input format of the int8 X-engine
 * (CORR_CI8): out[n_spectra][128][n_stream] (re, im) int8 pairs, code = clip(rint(S * scale), -127, 127) per component
 * (rint = round to nearest, ties to even; -128 is never produced.  The tensor-core kernel rounds ONCE -- S * scale is
 * formed and rounded to an integer by a single fused multiply-add on its fp32 sum S -- while the CUDA-core kernel rounds the
 * fp32 product first and then to an integer; the two can differ by one code only within an fp32 rounding error of a tie).  `scale` > 0 is the
 * caller's requantisation gain (e.g. 1 / (sigma_in * 16) * target sigma); `out` needs 2-byte alignment.  Everything
 * else as corr_fengine, the kernel choice included: the same stream counts and a 16-byte aligned `out` run on the
 * tensor cores (the rounding decision is taken on that kernel's fp32 sums), other geometries on the CUDA-core kernel.
 */
int corr_fengine_ci8(const void* in, void* out, int n_stream, long long n_spectra, float scale, void* stream);

/*
 * corr_xengine_static -- corr_xengine for callers that are not allowed to allocate device memory.
 *
 * Who needs it.  corr_create calls cudaMalloc (tile tables, the tile-feed counters), and corr_fengine / corr_xengine_host
 * allocate on first use.  Some users of a correlator library cannot make such a call at the point where they need a
 * result: a real-time capture process that has handed all of the GPU's memory to its own ring buffers at start-up and
 * must never see an allocation fail (or stall: cudaMalloc and cudaFree synchronise the whole device, which drops
 * samples on every other stream); a plug-in running inside a host application whose memory policy forbids driver
 * allocations after initialisation; a tool that attaches to a GPU which another tenant has already filled.  For them
 * this ONE entry point computes exactly what corr_create + corr_xengine compute (Eq. 2; lower
 * triangle with autocorrelations) and calls no cudaMalloc, cudaFree or other allocating CUDA routine, and
 * no malloc / new of its own, on any call.  There is no handle: the geometry is passed with every call.
 *
 * How.  It runs the CTA-pair tcgen05 kernel (CORR_KERNEL_PAIR).  The two things that kernel keeps in global memory
 * besides `in` and `out` -- the per-channel tile table and the 4-byte tile-feed counter -- live in a fixed array
 * compiled into the library, corr_static_scratch_bytes() = 16896 bytes.  Every GPU on which the process uses
 * libcorr.so holds that array from the moment the library's code is loaded onto it until the process exits, whether or
 * not this function is ever called.  The caller still owns and passes `in` and `out`.
 *
 *   n_station, n_pol, n_chan, n_time, dtype   as corr_create, with two limits of this entry point:
 *              n_station * n_pol <= CORR_STATIC_MAX_STREAMS (8192): the built-in tile table has room for the
 *              2080 tiles per channel of that size and no more; a larger problem is rejected with CORR_EINVAL and a
 *              message that names the limit (use corr_create / corr_xengine for it).
 *              n_station * n_pol * sample bytes must be a multiple of 16 (TMA addressing), else CORR_EUNSUPPORTED:
 *              the CUDA-core fallback of corr_xengine is not offered here.
 *   in, out, accumulate, stream               exactly as corr_xengine (DEVICE pointers, 16-byte aligned, same layouts
 *              and sizes: T*C*N*P*(2 or 4) bytes in, C*B*P*P*8 bytes out; asynchronous on `stream`).
 * Returns CORR_OK or a negative code; the message is corr_last_error(NULL).  All argument checks come before the
 * first CUDA call, so a rejected call touches no device.
 *
 * First call on a device.  The first successful call with a given device current does a one-time, host-side set-up
 * for that device (it looks up the array's device address, raises the kernel's shared-memory limit, queries how many
 * CTA pairs fit); it allocates nothing either, but it talks to the driver, so make that first call during start-up,
 * and before any stream capture is begun on that device.  Later calls only encode one tensor map on the host and
 * enqueue two kernels on `stream` (a small one that prepares the array, then the X-engine).
 *
 * Shared state -- read this.  Every call on a device uses the SAME array, and the array keeps what the last call left
 * in it; each call therefore re-initialises it (counter cleared, tile table rewritten) on its own stream before its
 * kernel starts.  Consequences: calls issued on ONE stream are safe back to back, with any mix of geometries; two
 * calls that can be in flight on the GPU at the same time (different streams without an event between them, or
 * several host threads of one process each calling it) race on the array and produce wrong visibilities without
 * any error.  Order them with events or use handles (each corr_create handle has its own scratch).  The host side is
 * thread-safe.
 *
 * CORR_CI8 overflow: a single call with n_time > 65535 returns CORR_EOVERFLOW; with accumulate != 0 there is no handle
 * to count the samples integrated so far, so keeping the running total within 65535 samples is the caller's job.
 */
#define CORR_STATIC_MAX_STREAMS 8192
int corr_xengine_static(int n_station, int n_pol, int n_chan, int n_time, int dtype, const void* in, void* out,
                        int accumulate, void* stream);
size_t corr_static_scratch_bytes(void);      /* size of the built-in scratch array, per GPU (16896) */

/* corr_destroy -- frees the handle and everything it owns.  NULL is a no-op. */
void corr_destroy(corr_handle h);

/* ---- helpers ------------------------------------------------------------------------------ */

size_t corr_input_bytes(corr_handle h);      /* T*C*N*P * (2 or 4); 0 for NULL  (C = n_chan_total of a window plan) */
size_t corr_output_bytes(corr_handle h);     /* C*B*P*P * 8;        0 for NULL                  */
long long corr_baseline_index(int i, int j); /* i(i+1)/2 + j for 0 <= j <= i, else -1           */

/* Message of the last failure on this handle (or, for NULL, of the last failed corr_create on this
 * thread).  The string is owned by the library and valid until the next call on the same handle. */
const char* corr_last_error(corr_handle h);

/* Force one of the CORR_KERNEL_* variants for subsequent corr_xengine calls (CORR_KERNEL_AUTO restores the
 * default choice).  CORR_EUNSUPPORTED if the geometry / device cannot run it.  corr_get_kernel returns the
 * kernel that WILL run (never CORR_KERNEL_AUTO): SIMT when TMA cannot address the geometry, else PAIR or SINGLE,
 * whichever executes the geometry cheaper (PAIR for 2*N*P >= 256 unless its 256 x 256 tiles pad a ragged 2*N*P by more
 * than 1.39x the 128-row tiles of SINGLE). */
int corr_set_kernel(corr_handle h, int kernel);
int corr_get_kernel(corr_handle h);

/* Which kernel corr_xengine will launch for this geometry: 1 = tcgen05 tensor-core kernel,
 * 0 = SIMT kernel (geometries whose per-channel sample row N*P*sample_bytes is not a multiple of 16
 * bytes -- N*P not a multiple of 8 (CI8) / 4 (CF16) -- where TMA box starts would be misaligned). */
int corr_uses_tensor_cores(corr_handle h);

/*
 * Corner turn (pre-X-engine data re-ordering; the GPU analogue of the paper's "indexing ... for
 * optimizing the GPU memory access"):
 *     ws    [c][m][t] = in[t][c][m]            (m = s*n_pol + p, complex kept interleaved)
 *     ws_rot[c][m][t] = (im, -re) of the same sample           (feeds the imaginary part)
 * with the time axis padded to corr_workspace_time(h) samples (zero filled).  CORR_CI8: -re saturates, so a real part
 * of -128 (outside the generators' [-127, 127]) becomes +127 in ws_rot; every other value is exact.
 *   in      DEVICE pointer as for corr_xengine.
 *   ws      DEVICE pointer, corr_workspace_bytes(h) bytes, 128-byte aligned: the two planes,
 *           ws then ws_rot, each n_chan * M * corr_workspace_time(h) samples.
 * Asynchronous on `stream`.  corr_xengine does NOT run it: its TMA feed reads `in` in place.
 */
int corr_corner_turn(corr_handle h, const void* in, void* ws, void* stream);
/* The same with a choice of planes: n_planes == 1 writes only `ws` (the first corr_workspace_bytes(h) / 2 bytes; a consumer
 * that forms the imaginary part without the rotated copy needs no more), n_planes == 2 is corr_corner_turn. */
int corr_corner_turn_planes(corr_handle h, const void* in, void* ws, int n_planes, void* stream);
size_t corr_workspace_bytes(corr_handle h);
int corr_workspace_time(corr_handle h);

/*
 * Introspection of the triangular tile schedule (host logic, no GPU work): writes up to `max_tiles`
 * entries of {row0, col0, ncols} (units: real components u = 2*m + {re:0, im:1} within a channel,
 * rows = conjugated side) for ONE channel and returns the number of tiles per channel.
 * Usable without a handle or a GPU.  `kernel` is CORR_KERNEL_SINGLE (128-row tiles, ncols <= 256) or
 * CORR_KERNEL_PAIR (256 x 256 tiles).
 */
int corr_tile_schedule(int n_station, int n_pol, int dtype, int kernel, int* tiles3, int max_tiles);

/* Number of kernels launched by the last corr_xengine / corr_xengine_host call on this handle (corr_xengine_host: one
 * per channel window). */
int corr_last_launch_count(corr_handle h);

#ifdef __cplusplus
}
#endif
#endif /* CORR_H_ */
