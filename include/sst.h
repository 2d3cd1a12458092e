/*
 * sst.h -- C ABI of libsst: B200-native unpacking + "three thresholds" clustering of
 * zero-suppressed silicon-strip FED data (arXiv 2101.11489).
 *
 * Problem statement: PAPER.md:25 (section 2: FED = 96 optical channels x 256 strips, CSR-like
 * zero-suppressed payload, per-strip calibration "e.g. gain and noise"), PAPER.md:31 (channel
 * location map, unpack to a structure of arrays), PAPER.md:33 (active strips, seed strips,
 * seed-index array, left/right boundaries, cluster charge vs cluster threshold; outputs: left
 * and right boundary, centroid, ADC values), PAPER.md:41 (several events in flight on CUDA
 * streams, pooled device memory).  Byte format, >= comparisons, gain formula, leftmost-seed
 * ownership and output order: BASELINE.json north_star / config 0 (DESIGN.md section 3 lists
 * every reading).
 *
 * Conventions
 *   - Plain C, no CUDA or torch types.  `stream` arguments are a cudaStream_t passed as void*.
 *   - "HOST" / "DEVICE" on every pointer says where the memory lives.  The caller owns every
 *     buffer it passes and keeps it alive until the work enqueued on `stream` has completed.
 *   - Global strip id g = (fed*96 + channel)*256 + strip.  N = n_feds*96*256.
 *   - Every call returns an sst_status.  Host-detectable errors enqueue nothing.  Problems only
 *     the device can see (malformed raw data, output capacity) are reported in
 *     sst_output.dev_status once the stream has completed.
 *   - After sst_upload_calib returns the context is read-only: sst_unpack_cluster may be called
 *     concurrently from several host threads on different streams.
 *   - CUDA graphs: once a stream has seen one plain call (which takes the stream's scratch from the
 *     pool), sst_unpack_cluster / sst_unpack_cluster_batch on that stream can be captured
 *     (cudaStreamBeginCapture) and the graph replayed: a launch is nothing but its parameters, the
 *     kernel keeps its work counter and the epoch of its FED words in device memory itself.
 *     The limits, because the graph holds the address of that stream's scratch: the plain call before
 *     the capture must have had at least as many events as the captured one (a capture that would
 *     have to allocate returns SST_ERR_INVALID_ARG and records nothing); after a capture the stream's
 *     scratch is never reallocated, so a later call on that stream with more events than it holds is
 *     refused with SST_ERR_INVALID_ARG; replay the graph on the captured stream only (or ordered
 *     with that stream's other work), one replay in flight at a time -- the replays share one work
 *     counter -- and never after sst_destroy.
 */
#ifndef SST_H
#define SST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SST_CHANNELS_PER_FED 96u
#define SST_STRIPS_PER_CHANNEL 256u
#define SST_STRIPS_PER_FED (96u * 256u)

typedef struct sst_ctx sst_ctx; /* opaque, owned by the library */

typedef enum {
    SST_OK = 0,
    SST_ERR_INVALID_ARG = 1, /* NULL pointer, n_feds == 0, threshold not finite or <= 0, ... */
    SST_ERR_CUDA = 2,        /* a CUDA call failed; sst_last_cuda_error() returns its code   */
    SST_ERR_NO_CALIB = 3,    /* sst_unpack_cluster before sst_upload_calib                   */
    SST_ERR_BAD_CALIB = 4,   /* gain/noise not finite or <= 0 at a non-bad strip; module map
                                decreasing, or a module crossing a FED boundary             */
    SST_ERR_TOO_LARGE = 5    /* sst_unpack_cluster_noalloc: the context's one-event scratch is larger
                                than SST_NOALLOC_SCRATCH_BYTES; nothing was enqueued        */
} sst_status;

typedef struct {
    uint32_t n_feds;               /* FEDs per event (fixed for the context)                    */
    int32_t device;                /* CUDA device ordinal                                       */
    uint32_t max_raw_bytes;        /* every DEVICE `raw` buffer holds at least this many readable
                                      bytes; a FED whose end offset exceeds it (or, in the HOST
                                      entry points, the event's raw_bytes) is flagged and empty */
    uint32_t max_events_in_flight; /* hint for the pool (0 = default 8)                         */
    uint32_t fed_strips_hint;      /* present (zero-suppressed) strips of a LARGE FED, e.g. the 99th
                                      percentile: sizes the per-FED shared-memory working set and
                                      with it the number of FEDs in flight per SM (when whole FEDs of
                                      that size would leave an SM fewer than 20 of them, the context is
                                      sized for FEDs worked on in pieces).  0 = derive it from
                                      max_raw_bytes / n_feds.  A FED above the hint is still processed
                                      correctly, in pieces or through a slower global-memory path   */
    uint32_t move_mode;            /* how the staged clusters reach their ordered place (same results):
                                      0 = inside sst_event_kernel, by the warps that find the FED work
                                      used up (one launch; launches that want the packed host block, hit
                                      coordinates or the compact SoA always take the second kernel);
                                      1 = always by sst_emit_kernel, launched behind it              */
    uint32_t trace;                /* 1 = launch the traced instantiations of sst_event_kernel: lane 0 of
                                      every warp adds the cycles of each phase of each FED and the
                                      launch's timeline to 32 words per stream (sst_trace_read); same
                                      results, ~7 % slower.  0 = no tracing code in the kernel at all  */
} sst_config; /* zero-initialise it: move_mode and trace must be 0 or 1, else sst_create returns
                 SST_ERR_INVALID_ARG */

/* S/N thresholds of the "three thresholds" algorithm: a strip is active at
 * adc/noise >= channel, a seed at adc/noise >= seed (both decided in exact arithmetic), a
 * cluster is accepted at charge/sqrt(sum noise^2) >= cluster. */
typedef struct { float channel, seed, cluster; } sst_thresholds;

/* dev_status words */
enum {
    SST_ST_FLAGS = 0,        /* SST_FLAG_* bits                                           */
    SST_ST_N_MALFORMED = 1,  /* channels whose run list is malformed (they contribute no strips) */
    SST_ST_N_CLUSTERS = 2,   /* clusters found (may exceed cap_clusters)                  */
    SST_ST_N_ADC = 3,        /* cluster ADC bytes found (may exceed cap_adc)              */
    SST_ST_N_OVERRUN = 4,    /* FEDs with bad offsets or a channel-length chain passing the FED end */
    SST_ST_N_SEEDS = 5,      /* seed strips found                                         */
    SST_ST_N_PRESENT = 6,    /* recorded strips with a non-zero ADC (when the compact SoA is
                                requested, else 0; may exceed cap_compact)                 */
    SST_ST_WORDS = 8
};
#define SST_FLAG_CLUSTER_CAP 1u /* more clusters than cap_clusters */
#define SST_FLAG_ADC_CAP 2u     /* more cluster ADC bytes than cap_adc */
#define SST_FLAG_MALFORMED 4u   /* >= 1 malformed channel */
#define SST_FLAG_OVERRUN 8u     /* >= 1 flagged FED */
#define SST_FLAG_COMPACT_CAP 16u /* more recorded strips than cap_compact */

/*
 * Output of one event.  All pointers are DEVICE pointers owned by the caller (HOST pointers
 * for sst_unpack_cluster_host).  Optional members may be NULL.
 *
 * Clusters are written in ascending global strip order of their first strip, i.e. ordered by
 * (module, first strip); cluster k has its gain-corrected ADCs at cl_adc[cl_adc_off[k] ..
 * + cl_width[k]) and cl_adc_off is the exclusive prefix sum of cl_width.
 * Capacity: cluster k is written iff k < cap_clusters and cl_adc_off[k]+cl_width[k] <= cap_adc;
 * the clusters written are always a prefix, *n_clusters is their number and nothing is written
 * beyond either capacity.  cap_clusters >= raw_bytes/2 and cap_adc >= raw_bytes never overflow
 * (a cluster costs at least two raw bytes: one ADC byte and an inactive strip or a run header
 * behind it; in zero-suppressed data, where every cluster is its own run, raw_bytes/3 suffices).
 */
typedef struct {
    uint8_t *strip_adc;   /* [N] dense unpacked ADC, absent strip = 0; NULL = do not materialise;
                             should be 16-byte aligned (else a slower store path is used)      */
    uint32_t *chan_off;   /* [n_feds*96] optional: byte offset in raw of the channel's first run */
    uint16_t *chan_len;   /* [n_feds*96] optional: payload length L of the channel               */
    uint32_t *seed_idx;   /* [cap_seeds] optional: ascending global ids of the seed strips       */
    uint32_t cap_seeds;
    uint32_t cap_clusters, cap_adc;
    uint32_t *n_clusters; /* [1] clusters written                                                */
    uint32_t *cl_module;  /* [cap_clusters] module id (as given in chan_module)                  */
    uint16_t *cl_first;   /* [cap_clusters] first strip, module-local (left boundary)           */
    uint16_t *cl_width;   /* [cap_clusters] strips in the cluster (right boundary = first+width-1) */
    int32_t *cl_charge;   /* [cap_clusters] sum of the gain-corrected ADCs                       */
    float *cl_bary;       /* [cap_clusters] barycenter, module-local strip units                 */
    uint32_t *cl_adc_off; /* [cap_clusters] offset of the cluster's ADCs in cl_adc               */
    float *cl_snr;        /* [cap_clusters] optional: charge / sqrt(sum noise^2)                 */
    uint8_t *cl_adc;      /* [cap_adc] gain-corrected ADCs min(254, floor(adc/gain + 0.5))       */
    uint32_t *dev_status; /* [SST_ST_WORDS], see above; fully written by every call              */
    /* Optional: the compact structure of arrays the paper's unpacker builds ("unpack
     * the data to SoA format", one entry per recorded strip) with the calibration
     * gathered per event: entry k is the k-th strip, in ascending global strip id,
     * whose dense ADC is non-zero.  All five arrays or none (compact_strip == NULL = not wanted);
     * entries beyond cap_compact are not written, dev_status[SST_ST_N_PRESENT] is the number
     * found.  DEVICE entry points only (sst_unpack_cluster, sst_unpack_cluster_batch): the HOST entry
     * points reject an sst_output that asks for them. */
    uint32_t *compact_strip; /* [cap_compact] global strip id                                    */
    uint8_t *compact_adc;    /* [cap_compact] raw ADC                                            */
    float *compact_noise;    /* [cap_compact] noise as uploaded                                  */
    float *compact_gain;     /* [cap_compact] gain as uploaded                                   */
    uint8_t *compact_bad;    /* [cap_compact] 1 = bad strip                                      */
    uint32_t cap_compact;
    /* Optional: global hit coordinates of the clusters ("convert clusters to global
     * hit coordinates in order to provide the necessary input for MKFIT"), from the geometry of
     * sst_upload_geometry: u = u0 + pitch * cl_bary; x = r cos(phi) - u sin(phi),
     * y = r sin(phi) + u cos(phi), z = z of the cluster's module, in float32 (absolute error
     * <= 1e-6 * max(|r|, |u|, |z|) against a double evaluation).  All three or none; NaN for a
     * module id >= n_modules or when no geometry was uploaded.  DEVICE entry points only. */
    float *hit_x, *hit_y, *hit_z; /* [cap_clusters] each */
} sst_output;

/* Creates a context on cfg->device: stream-ordered memory pool, calibration storage.
 * *out_ctx is NULL on failure. */
sst_status sst_create(const sst_config *cfg, sst_ctx **out_ctx);

/* Calibration upload, once.  HOST arrays: gain[N], noise[N] float32, bad[N]
 * (non-zero = bad strip, never active), chan_module[n_feds*96] = module id of every channel,
 * non-decreasing, equal ids = same module, a module never crosses a FED.  The arrays are
 * validated, copied to the device in an internal layout and may be freed on return (the call
 * synchronises).  The internal layout holds, per strip, the noise (+inf at bad strips) and a gain
 * FACTOR with which one fused multiply-add reproduces min(254, floor(adc / gain + 0.5)) of the
 * float32 division for every adc in 1..255: the call searches and verifies it per strip on all
 * host cores (~5 core-seconds for 10.8 M strips); strips without such a factor keep their gain
 * and are divided on the device.  Must not run concurrently with sst_unpack_cluster on the same
 * context. */
sst_status sst_upload_calib(sst_ctx *ctx, const float *gain, const float *noise, const uint8_t *bad,
                            const uint32_t *chan_module);

/* Module geometry for the hit conversion, once: HOST geom[n_modules*6] float32 =
 * {pitch, u0, r, cos phi, sin phi, z} of module id 0..n_modules-1 (module ids as given in
 * chan_module; reading s23: the paper gives no geometry, this flat-sensor model is the
 * build's own).  Copied before return; must not run concurrently with sst_unpack_cluster. */
sst_status sst_upload_geometry(sst_ctx *ctx, const float *geom, uint32_t n_modules);

/* One event: channel-location map, unpack, active/seed flags, seed expansion with
 * leftmost-seed ownership, gain correction, cluster threshold, ordered output
 * (PAPER.md:31,33).  raw: DEVICE, 16-byte aligned, >= cfg.max_raw_bytes readable bytes;
 * fed_offsets: DEVICE [n_feds+1] byte offsets of the FEDs in raw (16-byte multiples for the
 * fast path; the offsets must not step back: a FED with start > end, end > cfg.max_raw_bytes or a
 * start below any earlier entry of fed_offsets is flagged and empty).  thr and
 * out are HOST structs read before the call returns.  The work is enqueued on `stream` as ONE
 * kernel launch (sst_event_kernel: unpack + cluster per FED, then the ordered move of the clusters
 * by the warps that run out of FEDs) when cfg.move_mode is 0 and `out` asks for neither the compact
 * SoA nor hit coordinates, else as two (sst_emit_kernel does the move behind it); the call
 * does not synchronise.  Scratch comes from the context's
 * stream-ordered pool: one block per stream, allocated on the stream's first event and reused
 * (so a stream must not be driven by two host threads at once). */
sst_status sst_unpack_cluster(sst_ctx *ctx, const uint8_t *raw, const uint32_t *fed_offsets,
                              const sst_thresholds *thr, const sst_output *out, void *stream);

/* n_events independent events in one call (several events in flight): event e
 * belongs to streams[e % n_streams] with raw[e], fed_offsets[e] (DEVICE) and outs[e].  The events
 * share kernel launches (up to sst_info.events_per_launch events each, walked FED by FED so that
 * they share the calibration in L2): a launch runs on the first stream of its group after that
 * stream has waited (by CUDA event) for whatever the group's other streams had enqueued, and
 * those streams wait for the launch in turn -- so every event's inputs are honoured and its
 * result is complete in stream order on its own stream.  The streams thus only ORDER the events'
 * inputs and results; they add no concurrency: all events of a group run in one launch on one
 * stream.  Every event's result is exactly what sst_unpack_cluster gives.  raw, fed_offsets, outs and streams are HOST arrays read before the
 * call returns.  Does not synchronise. */
sst_status sst_unpack_cluster_batch(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                    const uint32_t *const *fed_offsets, const sst_thresholds *thr,
                                    const sst_output *outs, void *const *streams, uint32_t n_streams);

/* One event WITHOUT any allocation at call time: same arguments, same kernels and bit-for-bit the
 * same results as sst_unpack_cluster, but the scratch the kernels need between their
 * phases (work counter, per-FED totals, staged clusters, slow-path lists) is a fixed array compiled
 * into the library instead of a block taken from the context's pool on the stream's first event.
 *
 * Who needs it: code that must not reach the CUDA allocator once it is running.  Trigger and
 * data-acquisition loops fix their device-memory budget at start-up and cannot afford an allocation
 * that may stall the device, fail half-way through a run or grow the process's footprint; so do hosts
 * that have handed all device memory to an allocator of their own and plug-ins that run where the
 * embedding framework forbids allocation calls.  sst_unpack_cluster's first event on a new stream
 * (and any larger batch later) calls cudaMallocFromPoolAsync; this entry point never calls cudaMalloc,
 * cudaFree, their Async/pool forms or any library routine that allocates -- only cudaSetDevice, one
 * cudaMemsetAsync and the kernel launches.  raw, fed_offsets and every array of `out` are still the
 * caller's DEVICE buffers; the context (sst_create, sst_upload_calib: both allocate) is set up before.
 *
 * The price and the limit:
 *   - The array is SST_NOALLOC_SCRATCH_BYTES (32 MiB) of device memory that every GPU on which the
 *     library's kernels are loaded holds until the process exits, whether or not this call is used.
 *   - A context fits when the scratch of ONE event does: about 26 bytes per byte of
 *     cfg.max_raw_bytes plus 200 bytes per FED, i.e. a 440-FED detector with max_raw_bytes up to
 *     ~1.3 MB (one full-detector event of BASELINE.json config 1).  A larger context is refused with
 *     SST_ERR_TOO_LARGE before anything is enqueued.  One event per call; no batch form.
 *   - There is ONE array per GPU, shared by every context, stream and host thread of the process, and
 *     it keeps whatever the last call left in it.  Each call therefore first clears, on `stream`, the
 *     part that has to start at zero (work counter and per-FED words).  Two calls whose GPU work can
 *     overlap -- different streams, different contexts, different host threads -- RACE on it and give
 *     wrong results: keep all calls of a GPU on one stream, or order them with events.  The other
 *     entry points use pool scratch and may run beside it.
 *   - The FIRST call on each GPU looks up the array's device address (cudaGetSymbolAddress, with that
 *     GPU current), keeps it, and has the runtime load the kernels the entry point can launch; make
 *     that first call during set-up, before any stream capture begins.
 *   - A context created with trace = 1 is accepted but this call is never traced. */
#define SST_NOALLOC_SCRATCH_BYTES (32u << 20)
sst_status sst_unpack_cluster_noalloc(sst_ctx *ctx, const uint8_t *raw, const uint32_t *fed_offsets,
                                      const sst_thresholds *thr, const sst_output *out, void *stream);

/* The same event with HOST buffers: raw[raw_bytes] and fed_offsets[n_feds+1] are copied to
 * pooled device buffers on `stream`, the event is processed, and dev_status, n_clusters and the
 * cluster arrays (exactly n_clusters / n_adc elements; strip_adc, chan_off, chan_len, seed_idx
 * too when non-NULL) are copied back into the HOST arrays of `out`.  The call returns after
 * the stream has completed.  Pinned host memory makes the copies asynchronous to other streams. */
sst_status sst_unpack_cluster_host(sst_ctx *ctx, const uint8_t *raw, uint32_t raw_bytes,
                                   const uint32_t *fed_offsets, const sst_thresholds *thr,
                                   const sst_output *out, void *stream);

/* n_events events with HOST buffers in one call (transfers of some events overlap the
 * kernels of others): the events are cut into small chunks, chunk c is uploaded, processed in one
 * launch and read back on streams[c % n_streams] (use >= 3 streams for full overlap).  raw[e]
 * (raw_bytes[e] bytes), fed_offsets[e] and every array of outs[e] are HOST pointers.  When an
 * event's status and cluster arrays are pinned (mapped) host memory the kernels write them
 * directly over PCIe; otherwise they are staged in pooled device memory and copied back exactly
 * sized.  Results are as for sst_unpack_cluster_host.  Returns after all the streams it used have
 * completed. */
sst_status sst_unpack_cluster_host_batch(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                         const uint32_t *raw_bytes, const uint32_t *const *fed_offsets,
                                         const sst_thresholds *thr, const sst_output *outs, void *const *streams,
                                         uint32_t n_streams);

/* The host entry point with PACKED results: one download per event instead of one per array.
 * results[e].block is a HOST block (pinned for asynchronous copies) of at least
 * 64 + 20*cap_clusters + cap_adc bytes; on return it holds {dev_status[8], n_clusters, pad to 64
 * bytes} followed by the arrays cl_module, cl_charge, cl_bary, cl_adc_off (4 bytes per cluster),
 * cl_first, cl_width (2 bytes) and cl_adc back to back, each with K = min(clusters found,
 * cap_clusters) elements, and results[e].view is an sst_output whose HOST pointers point into the
 * block (strip_adc, chan_off, chan_len, seed_idx, cl_snr are not produced: NULL).  Events are
 * chunked over the streams as in sst_unpack_cluster_host_batch; returns when all are done. */
typedef struct {
    void *block;          /* HOST, caller-owned */
    uint64_t block_bytes; /* its size */
    sst_output view;      /* filled by the call */
} sst_packed_result;
sst_status sst_unpack_cluster_host_packed(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                          const uint32_t *raw_bytes, const uint32_t *const *fed_offsets,
                                          const sst_thresholds *thr, uint32_t cap_clusters, uint32_t cap_adc,
                                          sst_packed_result *results, void *const *streams, uint32_t n_streams);

/* Stream-ordered allocation of per-event buffers from the context's pool (cudaMallocAsync;
 * replaces the caching allocator of PAPER.md:41).  The pointer is usable by work enqueued on
 * `stream` after the call; free it with sst_event_free on a stream that has seen all its uses. */
sst_status sst_event_alloc(sst_ctx *ctx, uint64_t bytes, void *stream, void **out_ptr);
sst_status sst_event_free(sst_ctx *ctx, void *ptr, void *stream);

/* Stages one event: allocates pooled DEVICE buffers of cfg.max_raw_bytes and (n_feds+1)*4 bytes
 * on `stream` and enqueues the host-to-device copies of raw[raw_bytes] and fed_offsets[n_feds+1]
 * (HOST; pinned memory lets the copy overlap kernels of other streams).  Returns
 * the device pointers for sst_unpack_cluster on the same stream; release both with
 * sst_event_free.  Does not synchronise: the host arrays must stay valid until the copies ran. */
sst_status sst_event_upload(sst_ctx *ctx, const uint8_t *raw, uint32_t raw_bytes,
                            const uint32_t *fed_offsets, void *stream, uint8_t **d_raw,
                            uint32_t **d_fed_offsets);

/* Enqueues the device-to-host copy of `bytes` bytes from a DEVICE buffer (an output of
 * sst_unpack_cluster, e.g. one carved out of an sst_event_alloc block) into HOST memory on
 * `stream` (transfers of one event overlap the kernels of the others when dst is
 * pinned).  Does not synchronise: dst is valid once the stream has completed. */
sst_status sst_event_download(sst_ctx *ctx, void *dst, const void *src, uint64_t bytes, void *stream);

/* Synchronises the device and frees everything the context owns. */
sst_status sst_destroy(sst_ctx *ctx);

/* The cudaError_t of the last failed CUDA call on this context (0 if none). */
int32_t sst_last_cuda_error(const sst_ctx *ctx);
const char *sst_status_string(sst_status s);

/* Static facts about the compiled kernel and this context, for benchmarks: bytes of dynamic
 * shared memory per CTA of sst_event_kernel (a CTA is threads/32 independent warps, one FED at a
 * time each), threads per CTA, resident CTAs per SM as reported by the occupancy API, SM count,
 * kernels per launch with plain outputs (1; 2 with move_mode 1: sst_event_kernel + sst_emit_kernel),
 * the part of a warp's shared memory that holds a FED's payload and lists, events one launch can
 * take. */
typedef struct {
    uint32_t smem_bytes, threads, ctas_per_sm, sm_count, kernels_per_event, slot_bytes, events_per_launch;
    uint32_t pieces; /* 1: the slot was sized for whole FEDs; > 1: for FEDs worked on in that many pieces */
} sst_info;
sst_status sst_get_info(const sst_ctx *ctx, sst_info *info);

/* Tracing (contexts created with trace = 1).  Waits for `stream`, copies the stream's 32 trace words
 * to HOST `out` and clears them; SST_ERR_INVALID_ARG without tracing or before the stream's first
 * launch.  Words (sums over all FEDs of all launches of the stream since the last read):
 *   [0]  FEDs worked on
 *   [1..12] clock64 cycles of lane 0 per phase: 1 ticket + prologue, 2 payload staging (TMA wait),
 *        3 length chain, 4 pass 1 + scan (+ piece planning), 5 pass 2, 6 expansion (+ compact staging),
 *        7 dense SoA, 8 sweep, 9 members and heads, 10 counts + cluster list, 11 staging of the clusters,
 *        12 publish
 *   [13] FEDs moved inside sst_event_kernel, [14] cycles of those moves
 *   [20..23] %globaltimer nanoseconds of the LAST launch read: first warp started, first warp out of
 *        FED tickets, last warp out of FED tickets, last warp done (kernel end)
 * The rest is 0. */
#define SST_TRACE_WORDS 32
sst_status sst_trace_read(sst_ctx *ctx, void *stream, uint64_t *out);

#ifdef __cplusplus
}
#endif
#endif /* SST_H */
