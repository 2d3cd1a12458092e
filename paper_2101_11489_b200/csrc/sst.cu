// sst.cu -- libsst: unpack + three-threshold clustering of strip-tracker FED data on B200.
//
// ONE WARP PER FED (a FED is 96 channels x 256 strips; modules never cross a FED,
// DESIGN.md reading s10), one kernel launch per batch of up to 64 events.
//
// sst_event_kernel: a CTA is up to eight independent warps, each with a ~7 KB shared-memory slot,
// so 32 FEDs are in flight per SM and the serial parts of the method (the channel-length chain,
// the run headers) of one FED hide behind the parallel parts of the others; there is no
// block-wide barrier anywhere.  Warps draw (FED, event) tickets in FED-major order, so the FED's
// slab of the calibration is read from HBM once per launch (bulk-prefetched into L2 two FEDs ahead)
// and serves all the launch's events from L2.
// Per FED, everything after the unpack runs in the COMPACT index space of the FED's present
// strips (the structure of arrays of PAPER.md:31 has one entry per recorded strip):
//
//   a1 channel-location map : TMA bulk copy of the FED payload into the slot, the 96-step length
//                             chain walked in shared memory (PAPER.md:31 builds it on the CPU)
//   a2 unpack               : lane per channel, run HEADERS only: pass 1 validates and counts, a
//                             warp scan gives every channel its place in the lists, pass 2 writes the
//                             list entry of every run's first strip; then lane per ENTRY: a ballot
//                             finds each entry's run, its strip id and payload address follow, and
//                             the ADC list is the payload squeezed in place.  The dense SoA is put
//                             together in a 2 KB shared-memory window that leaves by TMA bulk store
//   a3-a6 sweep             : lane per CHUNK of consecutive entries, walked serially: one 8-byte
//                             gather of {noise, gain factor}, exact >= tests, link to the previous
//                             entry, q = min(254, floor(adc/gain + .5)) (one FMA with a factor
//                             verified per strip at upload to reproduce the float32 division), and
//                             the open candidate's (charge, sum noise^2 in double left to right,
//                             seed) in registers; a candidate is tested where it ends (leftmost-seed
//                             ownership is implicit: one test per maximal run).  Results are bits
//                             (links, seeds, ends of accepted clusters) kept in registers and
//                             flushed by all lanes together; a bit smear turns ends into members
//   a4 seed-index array     : seed mask + ordered compaction; materialised on request
//   a7 ordered output, 1/2  : counts by popcount scan, cluster records built lane per cluster and
//                             staged FED-locally in global scratch, FED totals in one 64-bit word
//                             tagged with the launch's epoch (release)
//   compact SoA (request)   : the FED's lists staged as they are
//
// A FED whose lists do not fit the slot is worked on in PIECES (channel ranges that start at module
// boundaries, sst_event_kernel<true>: contexts whose FEDs are large keep their warps per SM that
// way), or, when even that fails, through a pooled global scratch.
//
// a7, 2/2, the ordered move: a warp that finds the FED tickets used up goes on to MOVE staged FEDs
// -- exclusive prefix of the state words of the FED's predecessors (acquire), the staged FED into
// its free slot by TMA bulk copies, the cluster arrays streamed out in (module, first strip) order
// -- while the last FEDs are still being worked on by others.  Launches that want the packed host
// block, the clusters' global hit coordinates or the compact SoA with the calibration
// gathered per entry, and contexts with move_mode 1, take sst_emit_kernel behind
// sst_event_kernel on the same stream instead: one warp per (event, FED), no waiting.
// No tensor cores: nothing here is a contraction.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "sst.h"

namespace {

constexpr int kChan = 96;
constexpr int kStrip = 256;
constexpr int kFedStrips = kChan * kStrip;  // 24576
constexpr int kMaxEv = 64;        // events per launch
constexpr int kWarpsPerCta = 8;   // most warps (= FEDs in flight) per CTA, each with its own slot
constexpr int kMinCtas = 4;       // resident CTAs the register budget is set for (64 registers)
constexpr int kEmitCtas = 8;      // the same for sst_emit_kernel (CTAs of 4 warps)
constexpr uint32_t kHostChunk = 4;       // events per launch of the HOST entry points
constexpr uint32_t kFull = 0xffffffffu;
constexpr uint32_t kMaxFeds = 4096;
constexpr uint32_t kTabBytes = ((kChan + 1) * 4 + kChan * 2 + 15) & ~15;  // channel table of the FED, at the slot's end
constexpr uint32_t kFrameBytes = (3 * kChan + 16) * 4;  // what a FED in pieces keeps in its slot from piece to piece
constexpr uint32_t kWarpHdr = 16;        // mbarrier in front of a warp's slot
constexpr uint32_t kTailPad = 16;        // readable bytes behind the slot
constexpr uint32_t kSlabAhead = 2;       // FEDs between a calibration slab prefetch and its use
constexpr uint32_t kSlabMinEvents = 16;  // launches with fewer events prefetch the calibration per list entry instead

// FED aggregate, one 64-bit word per (event, FED), written by sst_event_kernel and read by
// sst_emit_kernel: overrun << 51 | malformed channels (7) << 44 | seeds (15) << 29 | cluster ADC
// bytes (15) << 14 | clusters (14).
// Bits 52..63 carry the launch's epoch (1..4095): a word counts as published by THIS launch only
// with the right tag, which is what the in-kernel move (below) waits for.
constexpr int kShOver = 51, kShMalf = 44, kShSeed = 29, kShAdc = 14, kShEpoch = 52;
constexpr uint32_t kEpochs = 4095;

struct EventDesc {
    const uint8_t *raw;
    const uint32_t *fed_offsets;
    uint8_t *packed;  // result block of the packed host entry point (else NULL): see emit kernel
    uint32_t raw_limit;  // readable bytes of raw: a FED ending beyond it is flagged and empty
    sst_output out;
};

struct KParams {
    const float2 *calib;     // {noise (+inf at bad strips), gain factor (see gain_apply)} per strip
    const uint2 *chan_info;  // {module id, first channel | end channel << 8 of the module}
    const float2 *calib_orig;  // {noise, gain} as uploaded (the compact SoA reports these)
    const uint8_t *bad;        // bad flags as uploaded
    const float *geom;         // [n_geom][6] {pitch, u0, r, cos phi, sin phi, z}, or NULL
    uint32_t n_geom;
    uint32_t *fed_present;     // [kMaxEv][n_feds] list entries << 16 | entries with a non-zero ADC (compact SoA)
    uint16_t *s_csid;          // staged list of a FED: strip ids and raw ADCs, for the compact SoA
    uint8_t *s_cadc;
    unsigned long long *fed_state;  // [kMaxEv][n_feds]
    unsigned long long *ticket;     // the stream's launch header: [0] ticket counter (0 when a launch starts: the last warp of
                                    // a launch to finish resets it), [1] warps finished, [2] launches so far modulo 4095
    unsigned long long *trace;      // 32 words of the stream's scratch (sst_trace_read), used by the traced kernels
    uint32_t state_words;  // words of fed_state (all events the scratch holds): cleared when the epoch starts over
    uint32_t move_chunk;  // clusters per bulk copy of the in-kernel move (from the slot size)
    uint32_t fused_move;  // 1: sst_event_kernel moves the staged clusters itself once its FED tickets are used up
    // global scratch of the slow path, one slice set per event
    uint16_t *g_strip;
    uint8_t *g_adc;
    uint32_t *g_rec;   // slow-path cluster lists (16-bit entries)
    uint32_t *g_mask;  // 4 arrays of g_mwords per event
    uint32_t g_ents, g_mwords;
    // staging of the FED-local results, read by sst_emit_kernel
    uint4 *s_rec;     // per accepted cluster {module, first | width << 16, charge, barycenter}
    uint32_t *s_off;  // offset of the cluster's ADCs inside its FED
    float *s_snr;
    uint8_t *s_adc;
    uint16_t *s_seed;
    uint32_t s_cl_stride;  // staged cluster slots per event
    double tcl2;
    float t_ch, t_seed;
    uint32_t max_raw_bytes, n_feds, n_events, slot_bytes;
    EventDesc ev[kMaxEv];
};

// The tag of this launch's FED aggregates, 1..4095: the stream's launch count (header word 2, kept
// by the kernel itself -- see the end of sst_event_kernel -- so that a launch is nothing but its
// parameters and can be captured in a CUDA graph and replayed) + 1.  Constant while a launch runs.
__device__ __forceinline__ uint32_t launch_epoch(const KParams &p) {
    return static_cast<uint32_t>(__ldg(p.ticket + 2)) + 1u;
}
// (every warp keeps it in the eight free bytes between its mbarrier and its slot)
__device__ __forceinline__ uint32_t warp_epoch(const uint8_t *slot) { return *reinterpret_cast<const uint32_t *>(slot - 8); }

// ------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_addr(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(unsigned long long *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE_%=;\n"
        "bra WAIT_LOOP_%=;\n"
        "WAIT_DONE_%=:\n"
        "}\n" ::"r"(smem_addr(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// TMA bulk copy global -> shared (non-tensor form), completion on an mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes,
                                         unsigned long long *bar, unsigned long long pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
            "r"(smem_addr(dst)),
        "l"(src), "r"(bytes), "r"(smem_addr(bar)), "l"(pol)
        : "memory");
}
// L2 residency.  The calibration (8 B per strip, 86.5 MB for 440 FEDs) is read by every event;
// the FED-major ticket order keeps the slabs in use hot, and raw data and outputs stream through
// once: calibration loads carry an evict_last policy, everything else that touches HBM
// evict_first.  (The persisting-L2 set-aside was measured slower and is not used.)
__device__ __forceinline__ unsigned long long policy_evict_last() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ unsigned long long policy_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// Calibration gather: nothing is reused through L1, and the line stays in L2 for the launch's
// other events (evict_last).
__device__ __forceinline__ float2 ld_calib(const float2 *p, unsigned long long pol) {
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(v.x), "=f"(v.y)
                 : "l"(p), "l"(pol));
    return v;
}
// streaming stores of the outputs
__device__ __forceinline__ void st_stream(uint8_t *p, uint32_t v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.u8 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_stream(uint16_t *p, uint32_t v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.u16 [%0], %1, %2;" ::"l"(p), "h"(static_cast<unsigned short>(v)), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_stream(uint32_t *p, uint32_t v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.u32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_stream(int32_t *p, int32_t v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.s32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_stream(float *p, float v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory");
}

// ------------------------------------------------------------------------------ arithmetic
// adc >= t * noise decided in exact arithmetic with float32 only: t*n = p + e exactly (FMA).
// noise = +inf (bad strip) gives p = inf, e = NaN -> false.
__device__ __forceinline__ bool ge_exact(float a, float t, float n) {
    const float p = __fmul_rn(t, n);
    const float e = __fmaf_rn(t, n, -p);
    return (a > p) | ((a == p) & (e <= 0.0f));
}
// min(254, floor(fl32(fl32(adc / gain) + 0.5)))  (IEEE RN division and add, no contraction)
__device__ __forceinline__ uint32_t gain_correct(float adc, float gain) {
    const float u = __fadd_rn(__fdiv_rn(adc, gain), 0.5f);
    const float fl = floorf(u);
    return fl >= 254.0f ? 254u : static_cast<uint32_t>(fl);
}

// The same through the strip's factor c from sst_upload_calib: c > 0 means
// min(254, floor(fma(adc, c, 0.5))) was checked there to equal gain_correct(adc, gain) for every
// adc 1..255 (c is 1/gain or a neighbour of it); c < 0 is -gain of a strip that has no such factor.
__device__ __forceinline__ uint32_t gain_apply(float adc, float c) {
    if (c > 0.0f) return min(254u, __float2uint_rz(__fmaf_rn(adc, c, 0.5f)));
    return gain_correct(adc, -c);
}

__device__ __forceinline__ unsigned long long warp_sum64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(kFull, v, d);
        if (lane >= d) v += u;
    }
    return v;
}
// ------------------------------------------------------------------------------ raw payload
// a1, generic path (payload not staged): the channel-length chain of one FED, checked as it goes.
__device__ __noinline__ bool walk_chain_checked(const uint8_t *rp, uint32_t fed_size, bool over, uint32_t *chan_off,
                                                uint16_t *chan_len) {
    uint32_t pos = 0;
    int c = 0;
    if (!over) {
#pragma unroll 1
        for (; c < kChan; ++c) {
            if (pos + 2 > fed_size) break;
            const uint32_t l16 = rp[pos] | (static_cast<uint32_t>(rp[pos + 1]) << 8);
            if (pos + 2 + l16 > fed_size) break;
            chan_off[c] = pos + 2;
            chan_len[c] = static_cast<uint16_t>(l16);
            pos += 2 + l16;
        }
    }
    over = c < kChan;
#pragma unroll 1
    for (; c < kChan; ++c) {  // channels behind an overrun are empty, recorded at the FED end
        chan_off[c] = fed_size;
        chan_len[c] = 0;
    }
    return over;
}

// a1, staged payload: the same chain walked speculatively by one lane -- no bounds checks inside
// the serial loop (reads are clamped into the slot), the 96 results are validated in parallel.
// It works on 32-bit shared-memory addresses: per channel one min, two byte loads, a multiply-add,
// an add and a store.  tab[c] = stage_addr + offset of the first run byte of channel c, c = 0..96
// (the lengths are differences).
__device__ __forceinline__ void walk_chain_speculative(uint32_t stage_addr, uint32_t clamp_addr, uint32_t tab_addr) {
    uint32_t pos = stage_addr + 2u;
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(tab_addr), "r"(pos) : "memory");
#pragma unroll 8
    for (int c = 0; c < kChan; ++c) {
        const uint32_t a = min(pos, clamp_addr);
        uint32_t lo, hi;
        asm volatile("ld.shared.u8 %0, [%1+-2];" : "=r"(lo) : "r"(a) : "memory");
        asm volatile("ld.shared.u8 %0, [%1+-1];" : "=r"(hi) : "r"(a) : "memory");
        pos = pos + 2u + (hi * 256u + lo);
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(tab_addr + 4u * static_cast<uint32_t>(c + 1)), "r"(pos) : "memory");
    }
}

// Tracing (sst_config.trace, kernel instantiations of their own): lane 0 of a warp adds the clock64
// cycles since its previous stamp to the slot of the phase that just ended, per FED.
enum { kTrFeds = 0, kTrMoved = 13, kTrMoveCycles = 14, kTrStart = 20, kTrFirstOut = 21, kTrLastOut = 22, kTrEnd = 23 };

struct FedCtx {
    uint32_t ev, f;
    uint32_t fo0;                  // the FED's start offset as given (reported in chan_off)
    uint32_t fed_start, fed_size;  // what is read: [fed_start, +fed_size), empty for a bad FED
    uint32_t overrun, n_malformed;
    uint32_t P;                    // present strips (list entries) of the FED
    uint32_t off[3], len[3];       // of channels lane, lane+32, lane+64
    uint32_t ebase[3];             // first list entry of those channels
    uint32_t opens;                // bit k: channel lane+32k opens a module
    // A FED whose lists do not fit the slot in one go is worked on in PIECES, channel ranges that
    // start at module boundaries, one after the other by the same warp (fed_size, P, off, len and
    // ebase then describe the piece; channels outside it have length 0):
    uint32_t ch_lo, ch_hi;         // the piece's channels [ch_lo, ch_hi); 0, 96 for a whole FED
    uint32_t last;                 // the piece ends the FED: the FED's word is published
    uint32_t cl_base, adc_base, seed_base, ent_base, nz_base;  // counts of the FED's earlier pieces
    long long t_prev;              // tracing: clock64 at the previous stamp
};

// slot k - 1 is the phase that ends where stamp k stands: 1 ticket + prologue, 2 payload staging,
// 3 chain, 4 pass 1 + scan, 5 pass 2, 6 expansion (+ compact staging), 7 dense SoA, 8 sweep,
// 9 members and heads, 10 counts + cluster list, 11 staging of the clusters, 12 publish (stamp 13)
__device__ __forceinline__ void trace_stamp(const KParams &p, FedCtx &c, const int lane, const int k) {
    if (lane == 0) {
        const long long t = clock64();
        atomicAdd(p.trace + (k - 1), static_cast<unsigned long long>(t - c.t_prev));
        c.t_prev = t;
    }
}

// a2 pass 1: a lane validates the run lists of its three channels (reading s2b) and
// counts their strips and runs, one channel after the other.  The loop body has no exit: a
// malformed channel is walked to its end like any other (every step advances by >= 3 bytes) and
// recognised afterwards.  A malformed channel contributes no strips (its length is zeroed).
__device__ __forceinline__ void scan_runs3(const uint8_t *rp, FedCtx &c, uint32_t (&cnt)[3], uint32_t (&runs)[3]) {
    uint32_t o0 = c.off[0], o1 = c.off[1], o2 = c.off[2], l0 = c.len[0], l1 = c.len[1], l2 = c.len[2];
    uint32_t n0 = 0, n1 = 0, n2 = 0, r0 = 0, r1 = 0, r2 = 0, okbits = 0;
#pragma unroll 1
    for (int k = 0; k < 3; ++k) {  // the register sets rotate
        uint32_t q = o0, nf = 0, r = 0;
        const uint32_t qe = o0 + l0;
        bool bad = false;
#pragma unroll 1
        while (q + 2u <= qe) {
            const uint32_t first = rp[q];
            uint32_t len = rp[q + 1];
            if (len == 0) len = 256;  // reading s2
            // a run that passes strip 255 leaves nf > 256: the next run (first <= 255) trips over
            // it here, the last one is caught below
            bad = bad || first < nf;
            nf = first + len;
            q += 2u + len;
            ++r;
        }
        __syncwarp();  // the lanes leave the walk at different times
        // truncated header, or run bytes passing the payload end: q != qe
        const bool ok = !bad && q == qe && nf <= static_cast<uint32_t>(kStrip);
        const uint32_t n = l0 - 2u * r;  // a well-formed channel of L bytes and r runs holds L - 2r strips
        o0 = o1; o1 = o2; l0 = l1; l1 = l2;
        n0 = n1; n1 = n2; n2 = ok ? n : 0u;
        r0 = r1; r1 = r2; r2 = ok ? r : 0u;
        okbits = (okbits >> 1) | (ok ? 4u : 0u);
    }
    cnt[0] = n0; cnt[1] = n1; cnt[2] = n2;
    runs[0] = r0; runs[1] = r1; runs[2] = r2;
    c.n_malformed = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const bool ok = (okbits >> k) & 1u;
        if (!ok) c.len[k] = 0;
        c.n_malformed += __popc(__ballot_sync(kFull, !ok));
    }
}

// Bits smeared towards lower entries along the links, inside one 32-entry word: bit e of the
// result is set iff some bit s >= e of x is set with link bits e+1 .. s all set (link bit i:
// entry i continues the candidate of entry i-1).  Five doubling steps.
__device__ __forceinline__ uint32_t smear_down(uint32_t x, uint32_t g) {
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
        x |= (x & g) >> s;
        g &= g << s;
    }
    return x;
}

// Cluster acceptance, the defining form (reading s15): Q^2 >= t_cl^2 * n2 with n2 the
// double sum of noise^2 over the candidate's strips taken strictly left to right (noise^2 is
// exact in double, so the fused multiply-add rounds exactly like a separate multiply and add).
// The noise is gathered again from the calibration: this runs only for candidates that cross a
// chunk boundary of the sweep and land within rounding distance of the threshold, and for the
// optional S/N output.
__device__ __noinline__ double n2_sequential(const float2 *cal, const uint16_t *strip_l, uint32_t head, uint32_t w) {
    double n2 = 0.0;
#pragma unroll 1
    for (uint32_t i = 0; i < w; ++i) {
        const double d = static_cast<double>(__ldg(&cal[strip_l[head + i] & 0x7fffu].x));
        n2 = __fma_rn(d, d, n2);
    }
    return n2;
}
__device__ __noinline__ bool accept_exact(const float2 *cal, const uint16_t *strip_l, uint32_t head, uint32_t w,
                                          uint32_t Q, double tcl2) {
    const double lhs = static_cast<double>(Q) * static_cast<double>(Q);
    return lhs >= __dmul_rn(tcl2, n2_sequential(cal, strip_l, head, w));
}
__device__ __noinline__ float snr_exact(const float2 *cal, const uint16_t *strip_l, uint32_t head, uint32_t w, int Q) {
    return static_cast<float>(static_cast<double>(Q) / sqrt(n2_sequential(cal, strip_l, head, w)));
}

// Fast-path layout of a warp's slot: offset of the strip-id list.  The payload (A bytes, the ADC
// list is squeezed into its first P16 bytes) is followed by a gap when the dense SoA is wanted, so
// that the 2048-byte window fits between the ADC list and the strip ids.
__device__ __forceinline__ uint32_t fast_strip_base(uint32_t A, uint32_t P16, bool want_dense) {
    return want_dense ? max(A, P16 + 2048u) : A;
}

// ------------------------------------------------------------------------------ lists -> clusters
// Everything after pass 1, by one warp, data-parallel over the FED's list of present strips (the
// structure of arrays of PAPER.md:31: one entry per recorded strip).  kFast: lists, masks and the
// candidate list live in the warp's shared-memory slot and the payload is staged there (the ADC
// list is the payload squeezed in place); else they live in this FED's slice of the global
// scratch and rp is whatever holds the payload.  Returns false (fast path only) when the cluster
// records outgrow the slot: the FED is then redone on the slow path (nothing has been published
// and every output written so far is rewritten identically).
template <bool kFast, bool kPiece, bool kTrace>
__device__ __forceinline__ bool fed_lists(const KParams &p, uint8_t *slot, const uint8_t *rp, FedCtx &c,
                                          const int lane, uint32_t &next_ticket) {
    const uint32_t f = c.f, P = c.P;
    // kPiece: c describes one piece of a FED (see FedCtx); else the whole FED, and all of this folds away
    const uint32_t ch_lo = kPiece ? c.ch_lo : 0u, ch_hi = kPiece ? c.ch_hi : static_cast<uint32_t>(kChan);
    const bool last = kPiece ? c.last != 0 : true;
    const uint32_t cl_base = kPiece ? c.cl_base : 0u, adc_base = kPiece ? c.adc_base : 0u, seed_base = kPiece ? c.seed_base : 0u,
                   ent_base = kPiece ? c.ent_base : 0u, nz_base = kPiece ? c.nz_base : 0u;
    const EventDesc &E = p.ev[c.ev];
    const sst_output &o = E.out;
    const uint32_t nw = (P + 31) >> 5;  // mask words in use; every mask has one more (zero) word
    const uint32_t lt = (1u << lane) - 1u, le = lt | (1u << lane);

    // per-channel constant of the payload address of an entry: src(e) = e + 2 * run(e) + ktab[channel]
    uint32_t *const ktab = reinterpret_cast<uint32_t *>(slot + p.slot_bytes - kTabBytes);
    uint16_t *strip_l;
    uint8_t *adc_l;
    // bit masks over the list entries: seeds; links, later heads of accepted clusters; ends, later
    // members of accepted clusters; per-word prefix counts
    uint32_t *mS, *mH, *mA, *mP;
    uint16_t *rec;              // list entries of the accepted clusters' first strips
    uint32_t rec_cap;
    uint8_t *window = nullptr;  // 2048 bytes for the dense SoA assembly, free once the lists are complete
    if (kFast) {
        // [0, A): the payload; the ADC list takes its place ([0, P)), the rest (grown by a gap to
        // 2048 bytes when the dense SoA is wanted) holds the window and then the cluster list.
        // Behind it the strip ids (2P bytes) and the masks.
        const uint32_t A = (c.fed_size + 15u) & ~15u, P16 = (P + 15u) & ~15u;
        const uint32_t S0 = fast_strip_base(A, P16, o.strip_adc != nullptr);
        adc_l = slot;
        strip_l = reinterpret_cast<uint16_t *>(slot + S0);
        mS = reinterpret_cast<uint32_t *>(slot + ((S0 + 2u * P + 15u) & ~15u));
        mH = mS + (nw + 2);
        mA = mH + (nw + 2);
        mP = mA + (nw + 2);
        rec = reinterpret_cast<uint16_t *>(slot + P16);
        rec_cap = (S0 - P16) / 2u;
        window = slot + P16;
    } else {
        const size_t eb = static_cast<size_t>(c.ev) * p.g_ents;
        const uint32_t slice = ((c.fed_start + 15u) & ~15u) + 16u * f;
        strip_l = p.g_strip + eb + slice;
        adc_l = p.g_adc + eb + slice;
        rec = reinterpret_cast<uint16_t *>(p.g_rec + eb + slice);
        mS = p.g_mask + static_cast<size_t>(c.ev) * 4u * p.g_mwords + (slice >> 5) + 4u * f;
        mH = mS + p.g_mwords;
        mA = mH + p.g_mwords;
        mP = mA + p.g_mwords;
        rec_cap = 0xffffffffu;
        // the slot is free up to the channel table unless the payload is staged in it
        const uint32_t A = (c.fed_size + 15u) & ~15u;
        if (rp != slot) window = slot;
        else if (A + 2048u + kTabBytes <= p.slot_bytes) window = slot + A;
    }
    const unsigned long long pol_last = policy_evict_last(), pol_first = policy_evict_first();
    uint8_t *const dense = o.strip_adc ? o.strip_adc + static_cast<size_t>(f) * kFedStrips : nullptr;
    const float2 *cal = p.calib + static_cast<size_t>(f) * kFedStrips;

    if (kTrace) trace_stamp(p, c, lane, 5);
    // ---------------------------------------------------------------- a2 pass 2: the run starts
    // Lane per channel again, headers only: the list entry of the first strip of every run gets
    // 1 + its strip id (bit 15 marks strip 0 of a channel that opens a module: nothing links across
    // it); all other entries stay zero.  Everything per strip is left to the expansion below.
    if (kFast) {
        uint4 *z = reinterpret_cast<uint4 *>(strip_l);  // 16-byte aligned; the masks behind it are not in use yet
#pragma unroll 1
        for (uint32_t i = lane; i * 8u < P; i += 32u) z[i] = make_uint4(0, 0, 0, 0);
    } else {
#pragma unroll 1
        for (uint32_t i = lane; i < P; i += 32u) strip_l[i] = 0;
    }
    __syncwarp();
    {
        uint32_t o0 = c.off[0], o1 = c.off[1], o2 = c.off[2], l0 = c.len[0], l1 = c.len[1], l2 = c.len[2];
        uint32_t b0 = c.ebase[0], b1 = c.ebase[1], b2 = c.ebase[2], opens = c.opens;
#pragma unroll 1
        for (int k = 0; k < 3; ++k) {
            uint32_t q = o0, e = b0;
            const uint32_t qe = o0 + l0;
            const uint32_t g1 = static_cast<uint32_t>(lane + 32 * k) * kStrip + 1u, open_bit = (opens & 1u) << 15;
#pragma unroll 1
            while (q < qe) {
                const uint32_t first = rp[q];
                uint32_t len = rp[q + 1];
                if (len == 0) len = 256;
                strip_l[e] = static_cast<uint16_t>(first == 0 ? (g1 | open_bit) : g1 + first);
                e += len;
                q += 2u + len;
            }
            __syncwarp();  // the lanes leave the walk at different times
            o0 = o1; o1 = o2; l0 = l1; l1 = l2; b0 = b1; b1 = b2; opens >>= 1;
        }
    }
    __syncwarp();

    if (kTrace) trace_stamp(p, c, lane, 6);
    // ---------------------------------------------------------------- a2: expansion, lane per entry
    // Entry e belongs to the last run that starts at or before it (the non-zero entries, by ballot):
    // its strip id is that run's first strip + the distance, and its ADC byte sits at e + 2 * (runs
    // up to it) + a per-channel constant in the payload (each earlier run costs two header bytes).
    // On the fast path the ADC list is written over the payload itself: an iteration reads at
    // addresses >= e + 4 and writes 32 bytes at e, after all its reads.
    {
        // In a FED without malformed channels or an overrun the per-channel constant is 2 * channel + 2
        // (two length bytes per channel up to and including the entry's own); else it is looked up.
        const bool regular = !kPiece && c.overrun == 0 && c.n_malformed == 0;
        const bool entry_prefetch = p.n_events < kSlabMinEvents;
        uint32_t run_before = 0, start_before = 0, v_before = 0;  // runs / last run start / its entry below this word
        const uint32_t last = P - 1u;                             // (P > 0 inside the loop)
        // two words of 32 entries per iteration, interleaved: the second word's carries follow from
        // the first word's ballot, everything else is independent (a warp is bound by the latency of
        // its own dependent steps, so two chains at once run nearly as fast as one)
        uint32_t vn_a = strip_l[min(static_cast<uint32_t>(lane), last)], vn_b = strip_l[min(static_cast<uint32_t>(lane) + 32u, last)];
        auto entry = [&](const uint32_t e, const uint32_t v, const uint32_t m, const uint32_t runs0, const uint32_t start0,
                         const uint32_t v0, uint32_t &sid, uint32_t &mark, uint32_t &a) {
            const uint32_t below = m & le;
            const uint32_t top = 31u - __clz(below);  // (-1 when below == 0: the shuffle result is then unused)
            const uint32_t vs = __shfl_sync(kFull, v, top);
            const uint32_t d = below ? lane - top : e - start0;  // distance to the run's first strip
            const uint32_t s0 = below ? vs : v0;
            sid = (s0 & 0x7fffu) - 1u + d;
            mark = d == 0 ? s0 & 0x8000u : 0u;
            const uint32_t r1 = runs0 + __popc(below);  // 1 + index of the entry's run
            const uint32_t ch = min(sid >> 8, static_cast<uint32_t>(kChan - 1));
            uint32_t kc = 2u * ch + 2u;
            if (!regular) kc = ktab[ch];
            a = rp[min(min(e, last) + 2u * r1 + kc, c.fed_size - 1u)];  // (clamped: lanes past the end)
        };
#pragma unroll 1
        for (uint32_t w = 0; w < nw; w += 2u) {
            const uint32_t e_a = w * 32u + lane, e_b = e_a + 32u;
            const bool in_a = e_a < P, in_b = e_b < P;
            const uint32_t v_a = in_a ? vn_a : 0u, v_b = in_b ? vn_b : 0u;
            vn_a = strip_l[min(e_a + 64u, last)];  // the next iteration's entries, ahead of their use
            vn_b = strip_l[min(e_b + 64u, last)];
            const uint32_t m_a = __ballot_sync(kFull, v_a != 0), m_b = __ballot_sync(kFull, v_b != 0);
            // carries into the second word
            const uint32_t mt_a = 31u - __clz(m_a), mt_b = 31u - __clz(m_b);
            const uint32_t va_top = __shfl_sync(kFull, v_a, mt_a), vb_top = __shfl_sync(kFull, v_b, mt_b);
            const uint32_t runs_b = run_before + __popc(m_a);
            const uint32_t start_b = m_a ? w * 32u + mt_a : start_before, v0_b = m_a ? va_top : v_before;
            uint32_t sid_a, sid_b, mark_a, mark_b, a_a, a_b;
            entry(e_a, v_a, m_a, run_before, start_before, v_before, sid_a, mark_a, a_a);
            entry(e_b, v_b, m_b, runs_b, start_b, v0_b, sid_b, mark_b, a_b);
            // a launch of few events cannot amortise a slab prefetch: the entry's calibration line is
            // requested now and arrives while the dense SoA is assembled
            if (entry_prefetch) {  // (uniform)
                if (in_a) asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(cal + sid_a));
                if (in_b) asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(cal + sid_b));
            }
            __syncwarp();  // all reads of both words before their writes
            if (in_a) {
                adc_l[e_a] = static_cast<uint8_t>(a_a);
                strip_l[e_a] = static_cast<uint16_t>(sid_a | mark_a);
            }
            if (in_b) {
                adc_l[e_b] = static_cast<uint8_t>(a_b);
                strip_l[e_b] = static_cast<uint16_t>(sid_b | mark_b);
            }
            run_before = runs_b + __popc(m_b);
            start_before = m_b ? (w + 1u) * 32u + mt_b : start_b;
            v_before = m_b ? vb_top : v0_b;
        }
    }
    __syncwarp();  // lists complete; the payload is dead from here on

    // ---------------------------------------------------------------- compact SoA, first half (on request)
    // the unpacker's product is a structure of arrays with one entry per recorded strip.
    // The FED's lists are exactly that; they are staged as they are (strip id, raw ADC) and
    // sst_emit_kernel moves them to their place in the event's arrays, adding the calibration.
    if (o.compact_strip) {
        const size_t cb = static_cast<size_t>(c.ev) * p.g_ents + c.fed_start + ent_base;
        uint32_t nz = 0;
#pragma unroll 1
        for (uint32_t i = lane; i < ((P + 31u) & ~31u); i += 32u) {
            uint32_t a = 0;
            if (i < P) {
                a = adc_l[i];
                p.s_csid[cb + i] = strip_l[i] & 0x7fffu;
                p.s_cadc[cb + i] = static_cast<uint8_t>(a);
            }
            nz += __popc(__ballot_sync(kFull, a != 0));
        }
        if (kPiece) {
            c.ent_base = ent_base + P;
            c.nz_base = nz_base + nz;
        }
        if (lane == 0 && last) p.fed_present[static_cast<size_t>(c.ev) * p.n_feds + f] = ((ent_base + P) << 16) | (nz_base + nz);
    }

    if (kTrace) trace_stamp(p, c, lane, 7);
    // ---------------------------------------------------------------- a2: dense SoA
    // The FED's 24576-byte block of the dense strip array is put together 2048 strips at a time
    // in a shared-memory window (zeros, then the present strips of the window from the sorted
    // lists) and leaves as one TMA bulk store per window: no zero-fill pass over HBM, no byte
    // scatter, and the way out costs the LSU pipe nothing.
    if (dense) {
        const uint32_t s_lo = ch_lo * kStrip, s_hi = ch_hi * kStrip;  // the piece's strips
        if ((reinterpret_cast<uintptr_t>(dense) & 15u) == 0 && window) {
            constexpr uint32_t kWin = 2048;
            uint4 *const win = reinterpret_cast<uint4 *>(window);
            uint32_t i0 = 0;  // first entry not yet placed
#pragma unroll
            for (uint32_t k = 0; k < kWin / 512u; ++k) win[lane + 32u * k] = make_uint4(0, 0, 0, 0);
#pragma unroll 1
            for (uint32_t base = s_lo; base < s_hi;) {
                __syncwarp();
                const uint32_t limit = kPiece ? min((base & ~(kWin - 1u)) + kWin, s_hi) : base + kWin;
                for (;;) {  // two consecutive entries per lane; the list is sorted by strip
                    const uint32_t i = i0 + 2u * lane;
                    const uint32_t ia = i < P ? i : 0u, ib = i + 1u < P ? i + 1u : 0u;  // loads stay in the lists
                    const uint32_t sa = strip_l[ia] & 0x7fffu, sb = strip_l[ib] & 0x7fffu;
                    const uint32_t va = adc_l[ia], vb = adc_l[ib];
                    const bool ina = i < P && sa < limit, inb = i + 1u < P && sb < limit;
                    if (ina) window[sa - base] = static_cast<uint8_t>(va);
                    if (inb) window[sb - base] = static_cast<uint8_t>(vb);
                    const uint32_t cnt = __popc(__ballot_sync(kFull, ina)) + __popc(__ballot_sync(kFull, inb));
                    i0 += cnt;
                    if (cnt < 64u) break;
                }
                // out: one TMA bulk store of the window by lane 0 (the generic-proxy writes of all lanes
                // are fenced first), then zeros again once the copy engine has read it
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) {
                    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dense + base),
                                 "r"(smem_addr(window)), "r"(limit - base), "l"(pol_first)
                                 : "memory");
                    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                }
                __syncwarp();
#pragma unroll
                for (uint32_t k = 0; k < kWin / 512u; ++k) win[lane + 32u * k] = make_uint4(0, 0, 0, 0);
                base = limit;
            }
        } else {  // unaligned output or no room for a window: bytes
#pragma unroll 1
            for (uint32_t b = s_lo + lane; b < s_hi; b += 32u) dense[b] = 0;
            __syncwarp();
#pragma unroll 1
            for (uint32_t i = lane; i < P; i += 32u) dense[strip_l[i] & 0x7fffu] = adc_l[i];
        }
        __syncwarp();
    }

    if (kTrace) trace_stamp(p, c, lane, 8);
    // ---------------------------------------------------------------- a3..a6: one sweep over the lists
    // Lane per CHUNK of consecutive entries, walked serially: active/seed tests, link to the previous
    // entry, and the running (charge, noise^2, seed) of the open candidate are thread-local, so a
    // candidate inside one chunk is decided exactly as the oracle does (double sum of noise^2,
    // left to right) with no cross-lane traffic.  What comes out are bits, collected in registers
    // for the 32-entry word the lane is in and flushed when it leaves the word: links, seeds, and
    // the last entries of accepted clusters.  A candidate that crosses a chunk boundary is put
    // together afterwards from the tail partial of one lane and the lead partials of the next lanes.
    uint32_t *const mL = mH, *const mE = mA;  // links become heads and ends become members further down
#pragma unroll 1
    for (uint32_t w = lane; w < nw + 2; w += 32) {
        mS[w] = 0;
        mL[w] = 0;
        mE[w] = 0;
    }
    const uint32_t Lc = ((P + 31u) >> 5) | 1u;  // odd: the lanes' list reads fall into different banks
    const bool want_seeds = o.seed_idx != nullptr;
    uint32_t n_seed_lane = 0;
    const uint32_t e0 = min(lane * Lc, P), e1 = min(e0 + Lc, P);
    {
        // is the entry before the chunk active?  (its raw ADC is read before any lane overwrites it)
        bool open = false;
        uint32_t prev_s = 0;
        if (e0 > 0) {
            const uint32_t sp = strip_l[e0 - 1], ap = adc_l[e0 - 1];
            prev_s = sp & 0x7fffu;
            if (ap) open = ge_exact(static_cast<float>(ap), p.t_ch, ld_calib(cal + prev_s, pol_last).x);
        }
        __syncwarp();
        bool lead = open;  // an open candidate at the chunk start began in an earlier chunk
        uint32_t hd = 0, Q = 0;
        double N = 0.0;
        bool seed = false;
        uint32_t lQ = 0, lEnd = 0;  // lead partial: the part of an earlier candidate inside this chunk
        double lN = 0.0;
        bool lSeed = false, lClosed = false;
        // Bits are collected per lane in CHUNK-local positions, 64 steps at a time, and shifted into
        // the masks by all lanes together (the step counter is uniform): links and seeds of the
        // step's entry, and "the candidate that ended with the PREVIOUS entry was accepted" -- the
        // end bits therefore sit one position high and are flushed one entry lower.
        uint32_t aL = 0, aE = 0, aS = 0;     // the 32 steps being filled
        uint32_t aL0 = 0, aE0 = 0, aS0 = 0;  // the 32 before them
        auto put = [&](uint32_t *m, uint32_t ebase, uint32_t lo, uint32_t hi) {  // local bit 0 = entry ebase
            const uint32_t wi = ebase >> 5, sh = ebase & 31u;
            const uint32_t w0 = lo << sh, w1 = __funnelshift_l(lo, hi, sh), w2 = sh ? hi >> (32u - sh) : 0u;
            if (w0) atomicOr(&m[wi], w0);
            if (w1) atomicOr(&m[wi + 1], w1);
            if (w2) atomicOr(&m[wi + 2], w2);
        };
        auto flush64 = [&](uint32_t ebase) {  // lower half in a?0, upper in a?
            put(mL, ebase, aL0, aL);
            if (ebase) put(mE, ebase - 1u, aE0, aE);
            else put(mE, 0u, __funnelshift_r(aE0, aE, 1), aE >> 1);  // (bit 0 is never set: nothing ends before entry 0)
            n_seed_lane += __popc(aS0) + __popc(aS);
            if (want_seeds) put(mS, ebase, aS0, aS);
            aL = aE = aS = aL0 = aE0 = aS0 = 0;
        };
        if (P) {  // (uniform)
            // software pipeline of depth one: the next entry's list reads and calibration gather
            // are issued before the current entry is worked on
            const uint32_t elast = min(max(e1, e0 + 1u), P) - 1u;
            // The lists of the fast path are addressed as 32-bit shared addresses the compiler cannot
            // re-derive (else it recomputes the warp's slot address, eleven instructions, at every
            // access inside the loop to save a register).
            uint32_t sl_sa = 0, al_sa = 0;
            if (kFast) {
                sl_sa = smem_addr(strip_l);
                al_sa = smem_addr(adc_l);
                asm volatile("" : "+r"(sl_sa), "+r"(al_sa));
            }
            auto ld_strip = [&](const uint32_t i) -> uint32_t {
                if (!kFast) return strip_l[i];
                uint32_t v;
                asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(sl_sa + 2u * i));
                return v;
            };
            auto ld_adc = [&](const uint32_t i) -> uint32_t {
                if (!kFast) return adc_l[i];
                uint32_t v;
                asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(al_sa + i));
                return v;
            };
            uint32_t sv_n = ld_strip(min(e0, P - 1u)), av_n = ld_adc(min(e0, P - 1u));
            float2 cv_n = ld_calib(cal + (sv_n & 0x7fffu), pol_last);
#pragma unroll 1
            for (uint32_t i0 = 0; i0 < Lc; i0 += 32u) {  // (uniform: every lane takes Lc steps, the last lanes idle in some)
                const uint32_t nsteps = min(32u, Lc - i0);
                uint32_t bit = 1u;
#pragma unroll 1
                for (uint32_t j = 0; j < nsteps; ++j, bit <<= 1) {
                    const uint32_t e = e0 + i0 + j;
                    const bool in = e < e1;
                    const uint32_t sv = sv_n, av = in ? av_n : 0u;
                    const float2 cv = cv_n;
                    {
                        const uint32_t en = min(e + 1u, elast);
                        sv_n = ld_strip(en);
                        av_n = ld_adc(en);
                        cv_n = ld_calib(cal + (sv_n & 0x7fffu), pol_last);
                    }
                    const uint32_t s15 = sv & 0x7fffu;
                    const float af = static_cast<float>(av);
                    const bool is_act = (av != 0) & ge_exact(af, p.t_ch, cv.x);
                    const bool is_seed = is_act & ge_exact(af, p.t_seed, cv.x);
                    // this entry continues the candidate of the previous one
                    const bool is_link = is_act & open & ((sv & 0x8000u) == 0) & (s15 == prev_s + 1u);
                    const bool ended = in & open & !is_link;  // the open candidate ended with entry e - 1
                    if (ended & lead) {  // (once per chunk at most)
                        lQ = Q; lN = N; lSeed = seed; lEnd = e - 1u; lClosed = true;
                    }
                    {
                        const double dq = static_cast<double>(Q);
                        const bool acc = ended & !lead & seed & (__dmul_rn(dq, dq) >= __dmul_rn(p.tcl2, N));
                        aE |= acc ? bit : 0u;
                    }
                    lead = lead & !ended;
                    if (is_act) {
                        if (!is_link) {
                            hd = e; Q = 0; N = 0.0; seed = false;
                        }
                        const uint32_t q = gain_apply(af, cv.y);
                        // kept for the staging
                        if (kFast) asm volatile("st.shared.u8 [%0], %1;" ::"r"(al_sa + e), "r"(q) : "memory");
                        else adc_l[e] = static_cast<uint8_t>(q);
                        Q += q;
                        const double d = static_cast<double>(cv.x);
                        N = __fma_rn(d, d, N);  // exact square, one rounding: the oracle's sum
                        seed = seed | is_seed;
                    }
                    aL |= is_link ? bit : 0u;
                    aS |= is_seed ? bit : 0u;
                    open = in ? is_act : open;
                    prev_s = in ? s15 : prev_s;
                }
                if (nsteps == 32u) {  // a full block of 32 steps: the first of a pair is set aside, the second flushed
                    if (i0 & 32u) {
                        flush64(e0 + i0 - 32u);
                    } else {
                        aL0 = aL; aE0 = aE; aS0 = aS;
                        aL = aE = aS = 0;
                    }
                }
            }
        }
        bool pend = false;  // an open candidate that began in this chunk and runs on
        if (open) {
            if (e1 == P) {  // the lists end here
                if (lead) {
                    lQ = Q; lN = N; lSeed = seed; lEnd = P - 1u; lClosed = true;
                } else if (seed) {
                    const double dq = static_cast<double>(Q);
                    if (__dmul_rn(dq, dq) >= __dmul_rn(p.tcl2, N)) atomicOr(&mE[(P - 1u) >> 5], 1u << ((P - 1u) & 31u));
                }
            } else if (lead) {  // the whole chunk lies inside a candidate of an earlier chunk
                lQ = Q; lN = N; lSeed = seed; lEnd = e1 - 1u; lClosed = false;
            } else {
                pend = true;
            }
        }
        {   // what is left in the registers: Lc = 64 k + r steps, r < 64
            const uint32_t r = Lc & 63u;
            if (r) {
                if (r < 32u) {  // only the lower half is in use, and it is still in the "being filled" set
                    aL0 = aL; aE0 = aE; aS0 = aS;
                    aL = aE = aS = 0;
                }
                flush64(e0 + (Lc - r));
            }
        }
        // candidates across chunk boundaries: tail + lead partials of the following lanes.  The sum
        // of partial sums is not the oracle's left-to-right sum; they differ by < (2w + 32) * 2^-53
        // relative, so the comparison is taken from it only outside that band.
        for (uint32_t dd = 1; __any_sync(kFull, pend); ++dd) {
            const uint32_t pk = __shfl_down_sync(kFull, lQ | (static_cast<uint32_t>(lSeed) << 30) |
                                                            (static_cast<uint32_t>(lClosed) << 31), dd);
            const uint32_t end_s = __shfl_down_sync(kFull, lEnd, dd);
            const double n_s = __shfl_down_sync(kFull, lN, dd);
            if (pend) {
                if (lane + dd > 31u) {
                    pend = false;  // cannot happen: the last lane's chunk ends the lists
                } else {
                    Q += pk & 0x3fffffffu;
                    N += n_s;
                    seed = seed || ((pk >> 30) & 1u);
                    if (pk >> 31) {
                        pend = false;
                        if (seed) {
                            const uint32_t wd = end_s - hd + 1u;
                            const double dq = static_cast<double>(Q);
                            const double lhs = __dmul_rn(dq, dq), rhs = __dmul_rn(p.tcl2, N);
                            bool acc;
                            if (fabs(lhs - rhs) > rhs * (static_cast<double>(wd + 16u) * 0x1p-51)) acc = lhs > rhs;
                            else acc = accept_exact(cal, strip_l, hd, wd, Q, p.tcl2);
                            if (acc) atomicOr(&mE[end_s >> 5], 1u << (end_s & 31u));
                        }
                    }
                }
            }
        }
    }
    __syncwarp();

    if (kTrace) trace_stamp(p, c, lane, 9);
    // ---------------------------------------------------------------- a5: members and heads
    // Lane per mask word: the end bits of the accepted clusters are smeared down along the links
    // (across word boundaries until nothing changes: a second round only happens for clusters
    // wider than a word), which gives the member mask; a member that is not linked is a head
    // (leftmost-seed ownership is implicit: one head per maximal run).
    {
        uint32_t carry_up = 0;  // (x & link & 1) of the word just above the group
#pragma unroll 1
        for (uint32_t g = (nw + 31u) >> 5; g-- > 0;) {  // groups of 32 words, from the top
            const uint32_t w = g * 32u + lane;
            const bool in = w < nw;
            const uint32_t lw = in ? mL[w] : 0u;
            uint32_t x = smear_down(in ? mE[w] : 0u, lw);
            for (;;) {
                uint32_t up = __shfl_down_sync(kFull, x & lw & 1u, 1);
                if (lane == 31) up = carry_up;
                const bool grow = up && !(x >> 31);
                if (grow) x = smear_down(x | 0x80000000u, lw);
                if (!__any_sync(kFull, grow)) break;
            }
            __syncwarp();
            if (in) {
                mA[w] = x;
                mH[w] = x & ~lw;
            }
            carry_up = __shfl_sync(kFull, x & lw & 1u, 0);
        }
    }
    __syncwarp();

    if (kTrace) trace_stamp(p, c, lane, 10);
    // ---------------------------------------------------------------- counts and cluster records
    // lane per mask word: exclusive prefix of (accepted heads, accepted members) per word, then
    // every head's list entry goes into the FED's cluster list, in order
    uint32_t fed_cl = 0, fed_adc = 0, fed_seed = 0;
    {
        uint32_t run = 0;  // heads << 16 | members
#pragma unroll 1
        for (uint32_t w0 = 0; w0 < nw; w0 += 32) {
            const uint32_t w = w0 + lane;
            uint32_t v = 0;
            if (w < nw) v = (__popc(mH[w]) << 16) | __popc(mA[w]);
            const uint32_t incl = warp_incl_scan(v, lane);
            if (w < nw) mP[w] = run + incl - v;
            run += __shfl_sync(kFull, incl, 31);
        }
        fed_seed = __reduce_add_sync(kFull, n_seed_lane);
        fed_cl = run >> 16;
        fed_adc = run & 0xffffu;
        if (kFast && fed_cl > rec_cap) return false;
        __syncwarp();
#pragma unroll 1
        for (uint32_t w = lane; w < nw; w += 32) {
            uint32_t mh = mH[w], k = mP[w] >> 16;
            while (mh) {
                const uint32_t b = __ffs(mh) - 1u;
                mh &= mh - 1u;
                rec[k++] = static_cast<uint16_t>(w * 32u + b);
            }
        }
    }
    __syncwarp();

    if (kTrace) trace_stamp(p, c, lane, 11);
    // ---------------------------------------------------------------- a7, first half: publish + stage
    // The FED's counts go into its state word; its clusters, cluster ADCs and seeds are staged in
    // FED-local order in global scratch.  sst_emit_kernel, launched behind this kernel on the same
    // stream, turns the counts into offsets and moves everything to its (module, first strip)
    // ordered place -- no warp ever waits for another one.
    const size_t sb = static_cast<size_t>(c.ev) * p.s_cl_stride + c.fed_start / 2u + f + cl_base;
    const size_t ab = static_cast<size_t>(c.ev) * p.g_ents + c.fed_start;
    // next FED of this warp: the ticket arrives while the staging runs
    if (lane == 0 && last) next_ticket = static_cast<uint32_t>(atomicAdd(p.ticket, 1ull));
    {
        // cluster records: lane per cluster, consecutive lanes write consecutive records
        const uint2 *cinfo = p.chan_info + static_cast<size_t>(f) * kChan;
        uint8_t *const sa = p.s_adc + ab;  // the FED's cluster ADCs, in order
#pragma unroll 1
        for (uint32_t k0 = 0; k0 < fed_cl; k0 += 32) {
            const uint32_t k = k0 + lane;
            const bool have = k < fed_cl;
            uint32_t hd = 0, wd = 0, off = 0;
            if (have) {
                hd = rec[k];
                const uint32_t wi = hd >> 5, b = hd & 31u;
                const uint32_t ma = mA[wi], mh = mH[wi];
                // its ADCs start behind those of the members before it
                off = adc_base + (mP[wi] & 0xffffu) + __popc(ma & ((1u << b) - 1u));
                // width: the members behind the head that are not heads themselves, 32 at a time
                const uint32_t v = __funnelshift_rc(ma & ~mh, mA[wi + 1] & ~mH[wi + 1], b + 1u);
                uint32_t n1 = __ffs(~v) - 1u;  // trailing ones
                if (v == kFull) {
                    n1 = 32;
                    for (;;) {  // (the zero words behind the masks end it)
                        const uint32_t e = hd + n1 + 1u;
                        if (!(((mA[e >> 5] & ~mH[e >> 5]) >> (e & 31u)) & 1u)) break;
                        ++n1;
                    }
                }
                wd = 1u + n1;
            }
            if (have) {
                const uint32_t st0 = strip_l[hd] & 0x7fffu;
                const uint2 cm = __ldg(cinfo + (st0 >> 8));  // in flight during the sums
                // The first four corrected ADCs in one word (two aligned loads of the list, which may be
                // read a few bytes past its end): charge and first moment as byte dot products, the
                // staged bytes from the same register.  Wider clusters (few) go on in a loop.
                uint32_t q4;
                {
                    const uint32_t *w = reinterpret_cast<const uint32_t *>(adc_l + (hd & ~3u));
                    q4 = __funnelshift_r(w[0], w[1], 8u * (hd & 3u));
                    if (wd < 4u) q4 &= (1u << (8u * wd)) - 1u;
                }
                int Q = __dp4a(q4, 0x01010101u, 0u), M = __dp4a(q4, 0x03020100u, 0u);  // M <= 254 * 768^2 / 2
                {
                    uint8_t *d = sa + off;  // neighbouring lanes write neighbouring bytes
                    d[0] = static_cast<uint8_t>(q4);
                    if (wd > 1u) d[1] = static_cast<uint8_t>(q4 >> 8);
                    if (wd > 2u) d[2] = static_cast<uint8_t>(q4 >> 16);
                    if (wd > 3u) d[3] = static_cast<uint8_t>(q4 >> 24);
                }
#pragma unroll 1
                for (uint32_t j = 4; j < wd; ++j) {
                    const int q = adc_l[hd + j];
                    Q += q;
                    M += static_cast<int>(j) * q;
                    sa[off + j] = static_cast<uint8_t>(q);
                }
                const uint32_t first = st0 - (cm.y & 0xffu) * kStrip;
                // barycenter in float32: first + M/Q is good to ~2e-7 relative (tolerance 1e-6)
                const float bary = __fadd_rn(static_cast<float>(first), __fdiv_rn(static_cast<float>(M), static_cast<float>(Q)));
                p.s_rec[sb + k] = make_uint4(cm.x, first | (wd << 16), static_cast<uint32_t>(Q), __float_as_uint(bary));
                p.s_off[sb + k] = off;
                if (o.cl_snr) p.s_snr[sb + k] = snr_exact(cal, strip_l, hd, wd, Q);
            }
        }
    }
    // a4: seed-index array (on request), FED-local strip ids
    if (o.seed_idx) {
        uint32_t k0 = 0;
#pragma unroll 1
        for (uint32_t w = 0; w < nw; ++w) {
            const uint32_t sw = mS[w];
            if ((sw >> lane) & 1u) p.s_seed[ab + seed_base + k0 + __popc(sw & lt)] = strip_l[w * 32u + lane] & 0x7fffu;
            k0 += __popc(sw);
        }
    }
    if (kPiece) {
        c.cl_base = cl_base + fed_cl;
        c.adc_base = adc_base + fed_adc;
        c.seed_base = seed_base + fed_seed;
    }
    if (kTrace) trace_stamp(p, c, lane, 12);
    if (!last) return true;  // (uniform) more pieces of this FED follow
    // publish: the FED's counts, tagged with the launch's epoch, behind everything staged above
    // (release: the in-kernel move of another warp may read the staging as soon as it sees the word,
    // and it reads it with TMA bulk copies: the writers order their generic-proxy stores before
    // async-proxy accesses)
    if (p.fused_move) asm volatile("fence.proxy.async.global;" ::: "memory");
    __syncwarp();
    if (lane == 0) {
        const unsigned long long v = (static_cast<unsigned long long>(warp_epoch(slot)) << kShEpoch) |
                                     (static_cast<unsigned long long>(c.overrun) << kShOver) |
                                     (static_cast<unsigned long long>(c.n_malformed) << kShMalf) |
                                     (static_cast<unsigned long long>(seed_base + fed_seed) << kShSeed) |
                                     (static_cast<unsigned long long>(adc_base + fed_adc) << kShAdc) | (cl_base + fed_cl);
        asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p.fed_state + static_cast<size_t>(c.ev) * p.n_feds + f), "l"(v) : "memory");
    }
    if (kTrace) {
        trace_stamp(p, c, lane, 13);
        if (lane == 0) atomicAdd(p.trace + kTrFeds, 1ull);
    }
    return true;
}

// ------------------------------------------------------------------------------ one FED, one warp
// Returns false when the FED has to be redone with force_slow (see fed_lists).
// kPieces: a FED whose lists do not fit the slot is worked on in pieces (contexts whose slot was
// sized for that); else it goes through the global scratch.
template <bool kPieces, bool kTrace>
__device__ __forceinline__ bool process_fed(const KParams &p, unsigned long long *mbar, uint8_t *slot,
                                            const uint32_t ticket, const int lane, const bool force_slow,
                                            uint32_t &mbar_phase, uint32_t &next_ticket) {
    FedCtx c;
    if (kTrace) c.t_prev = clock64();
    // FED-major order: the same FED of all the launch's events back to back, so the FED's slab of
    // the calibration (196 KB) is reused from L2 while it is hot
    c.f = ticket / p.n_events;
    c.ev = ticket - c.f * p.n_events;
    const uint32_t f = c.f;
    const EventDesc &E = p.ev[c.ev];
    const sst_output &o = E.out;
    // The first event of a FED streams the calibration slab of a FED a few places ahead into L2
    // (one bulk prefetch of 6 KB per lane): the launch's events then gather from L2, and HBM sees
    // sequential reads instead of the first-touch misses of scattered 8-byte loads.
    if (c.ev == 0 && p.n_events >= kSlabMinEvents && f + kSlabAhead < p.n_feds) {
        const uint8_t *slab = reinterpret_cast<const uint8_t *>(p.calib + static_cast<size_t>(f + kSlabAhead) * kFedStrips);
        constexpr uint32_t kPiece = kFedStrips * sizeof(float2) / 32;
        asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(slab + lane * kPiece), "r"(kPiece), "l"(policy_evict_last()) : "memory");
    }
    uint32_t *const chan_off = reinterpret_cast<uint32_t *>(slot + p.slot_bytes - kTabBytes);
    uint16_t *const chan_len = reinterpret_cast<uint16_t *>(chan_off + kChan + 1);

    if (kTrace) trace_stamp(p, c, lane, 2);
    // ---------------------------------------------------------------- a1: stage the FED payload
    // lanes 0/1 fetch the two offsets; lane 0 starts the bulk copy
    const uint32_t fo = lane < 2 ? E.fed_offsets[f + lane] : 0u;
    const uint32_t fo0 = __shfl_sync(kFull, fo, 0), fo1 = __shfl_sync(kFull, fo, 1);
    // (the bulk copy is started on the FED's own two offsets; reading s3c -- the offsets never step
    // back: a FED that starts below an earlier offset is flagged and empty -- is checked while it
    // is in flight, and a refused FED simply ignores what was copied)
    const bool valid0 = fo0 <= fo1 && fo1 <= E.raw_limit;
    c.fo0 = fo0;
    c.fed_start = valid0 ? fo0 : 0u;
    c.fed_size = valid0 ? fo1 - fo0 : 0u;
    const bool staged = c.fed_size + kTabBytes <= p.slot_bytes && ((c.fed_start | c.fed_size) & 15u) == 0 &&
                        (reinterpret_cast<uintptr_t>(E.raw) & 15u) == 0;
    __syncwarp();  // every lane is done with the slot of the previous FED
    const bool copying = staged && c.fed_size;
    if (copying && lane == 0) {
        fence_proxy_async();  // earlier generic-proxy accesses to the slot before the async write
        mbar_expect_tx(mbar, c.fed_size);
        bulk_g2s(slot, E.raw + c.fed_start, c.fed_size, mbar, policy_evict_first());
    }
    // the valid FEDs of an event are disjoint and ascending (the FED-local staging areas are keyed
    // by the start offset)
    uint32_t fo_max = 0;
#pragma unroll 1
    for (uint32_t j = lane; j < f; j += 32) fo_max = max(fo_max, E.fed_offsets[j]);
    fo_max = __reduce_max_sync(kFull, fo_max);
    const bool valid = valid0 && fo_max <= fo0;
    if (!valid) {
        c.fed_start = 0;
        c.fed_size = 0;
    }
    c.overrun = valid ? 0u : 1u;
    // meanwhile: fetch the module map
    c.opens = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t ch = lane + 32 * k;
        const uint2 ci = __ldg(p.chan_info + static_cast<size_t>(f) * kChan + ch);
        if ((ci.y & 0xffu) == ch) c.opens |= 1u << k;
    }
    const uint8_t *rp = staged ? slot : E.raw + c.fed_start;
    if (copying) {
        mbar_wait(mbar, mbar_phase);  // every lane waits: async-proxy writes visible to all readers
        mbar_phase ^= 1u;
    }

    if (kTrace) trace_stamp(p, c, lane, 3);
    // ---------------------------------------------------------------- a1: walk the length chain
    if (staged) {
        const uint32_t sa = smem_addr(slot);
        if (lane == 0) walk_chain_speculative(sa, sa + p.slot_bytes - kTabBytes, smem_addr(chan_off));
        __syncwarp();
        // validate the speculative chain: channels from the first bad one on are empty
        uint32_t bad = 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            c.off[k] = chan_off[lane + 32 * k] - sa;
            c.len[k] = (chan_off[lane + 32 * k + 1] - sa - c.off[k] - 2u) & 0xffffu;
            const bool ok = c.overrun == 0 && c.off[k] <= c.fed_size && c.off[k] + c.len[k] <= c.fed_size;
            const uint32_t m = ~__ballot_sync(kFull, ok);
            if (!bad && m) bad = 32u * k + __ffs(m);  // 1 + index of the first bad channel
        }
        if (bad) {
            c.overrun = 1;
#pragma unroll
            for (int k = 0; k < 3; ++k)
                if (static_cast<uint32_t>(lane + 32 * k) >= bad - 1u) {
                    c.off[k] = c.fed_size;
                    c.len[k] = 0;
                }
        }
    } else {
        uint32_t over = c.overrun;
        if (lane == 0) over = walk_chain_checked(rp, c.fed_size, c.overrun != 0, chan_off, chan_len) ? 1u : 0u;
        c.overrun = __shfl_sync(kFull, over, 0);
        __syncwarp();
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            c.off[k] = chan_off[lane + 32 * k];
            c.len[k] = chan_len[lane + 32 * k];
        }
    }
    __syncwarp();  // the channel table is in registers: its place in the slot is free

    if (kTrace) trace_stamp(p, c, lane, 4);
    // ---------------------------------------------------------------- a2 pass 1: run headers
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t ch = lane + 32 * k;
        if (o.chan_off) o.chan_off[f * kChan + ch] = c.fo0 + c.off[k];
        if (o.chan_len) o.chan_len[f * kChan + ch] = static_cast<uint16_t>(c.len[k]);
    }
    uint32_t cnt[3], runs[3];
    if (staged) scan_runs3(slot, c, cnt, runs);
    else scan_runs3(rp, c, cnt, runs);
    // exclusive scans of the 96 strip and run counts (one scan: runs in the upper half word)
    uint32_t tot = 0, exs[3];
    uint32_t *const ktab = chan_off;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t v = cnt[k] | (runs[k] << 16);
        const uint32_t inc = warp_incl_scan(v, lane);
        const uint32_t ex = tot + inc - v;
        exs[k] = ex;
        c.ebase[k] = ex & 0xffffu;
        // payload address of entry e of this channel: off + (e - ebase) + 2 * (run(e) - rbase + 1),
        // i.e. e + 2 * (runs up to and including its own) + this constant
        ktab[lane + 32 * k] = c.off[k] - (ex & 0xffffu) - 2u * (ex >> 16);
        tot += __shfl_sync(kFull, inc, 31);
    }
    c.P = tot & 0xffffu;  // present strips of the FED (<= 24576; the runs, <= 12288, sit in the upper half)
    c.ch_lo = 0;
    c.ch_hi = kChan;
    c.last = 1;
    c.cl_base = c.adc_base = c.seed_base = c.ent_base = c.nz_base = 0;
    __syncwarp();

    // fast path: window / cluster list, strip ids and masks fit behind the ADC list
    const bool want_dense = o.strip_adc != nullptr;
    auto fits_in = [&](const uint32_t bytes, const uint32_t strips, const uint32_t room) {
        const uint32_t A = (bytes + 15u) & ~15u, P16 = (strips + 15u) & ~15u;
        const uint32_t S0 = fast_strip_base(A, P16, want_dense);
        return ((S0 + 2u * strips + 15u) & ~15u) + 16u * (((strips + 31u) >> 5) + 2u) + kTabBytes <= room;
    };
    auto fits = [&](const uint32_t bytes, const uint32_t strips) { return fits_in(bytes, strips, p.slot_bytes); };
    // (a piece leaves room for the frame that carries the FED from piece to piece)
    auto fits_piece = [&](const uint32_t bytes, const uint32_t strips) { return fits_in(bytes, strips, p.slot_bytes - kFrameBytes); };
    // ---------------------------------------------------------------- a FED in pieces
    // When the lists of the whole FED do not fit the slot the warp works through it in up to seven
    // pieces, channel ranges that start where a module starts (nothing links across), each as
    // large as fits.  A piece's part of the payload is fetched again from global memory (it is
    // in L2) to the start of the slot; everything per channel is in registers already.
    // value of a per-channel quantity at boundary b (a channel index, or 96)
    auto at = [&](const uint32_t (&v)[3], const uint32_t b, const uint32_t at_end) {
        const uint32_t x0 = __shfl_sync(kFull, v[0], b & 31u), x1 = __shfl_sync(kFull, v[1], b & 31u),
                       x2 = __shfl_sync(kFull, v[2], b & 31u);
        return b >= static_cast<uint32_t>(kChan) ? at_end : b < 32u ? x0 : b < 64u ? x1 : x2;
    };
    bool slow = force_slow || !staged;
    unsigned long long plan = 0;  // boundaries, 8 bits each
    uint32_t n_pieces = 0;        // 0: the whole FED at once
    if (!kPieces) {
        slow = slow || !fits(c.fed_size, c.P);
    } else if (!slow && !fits(c.fed_size, c.P)) {  // (uniform)
        for (uint32_t lo = 0; lo < static_cast<uint32_t>(kChan);) {
            // (16-byte granules of the payload; an overrun FED is fetched to its end)
            const uint32_t g_lo = (at(c.off, lo, c.fed_size + 2u) - 2u) & ~15u, e_lo = at(exs, lo, tot) & 0xffffu;
            uint32_t best = 0;
            if (fits_piece(c.fed_size - g_lo, c.P - e_lo)) {
                best = kChan;
            } else {
#pragma unroll
                for (int k = 2; k >= 0; --k) {
                    const uint32_t ch = lane + 32 * k;
                    const uint32_t hi = c.overrun ? c.fed_size : (c.off[k] - 2u + 15u) & ~15u;
                    const bool ok = ch > lo && ((c.opens >> k) & 1u) && hi >= g_lo && fits_piece(hi - g_lo, (exs[k] & 0xffffu) - e_lo);
                    const uint32_t m = __ballot_sync(kFull, ok);
                    if (!best && m) best = 32u * k + 31u - __clz(m);
                }
            }
            if (!best || n_pieces == 7) {  // a module that does not fit, or too many pieces
                slow = true;
                break;
            }
            plan |= static_cast<unsigned long long>(best) << (8u * n_pieces);
            ++n_pieces;
            lo = best;
        }
    }
    if (slow) return fed_lists<false, false, kTrace>(p, slot, rp, c, lane, next_ticket);
    if (!kPieces || n_pieces == 0) return fed_lists<true, false, kTrace>(p, slot, slot, c, lane, next_ticket);
    // What the pieces need of the FED goes into a frame at the top of the slot (below the channel
    // table; piece 0 stays clear of it, the rest of the payload up there is fetched again anyway)
    // and comes back at the start of every piece: nothing of it stays in registers across a piece
    // (with ~150 bytes of spills per thread and no L1 to speak of beside 229 KB of shared memory,
    // every spilled value would come back from L2).
    uint32_t *const fr = reinterpret_cast<uint32_t *>(slot + p.slot_bytes - kTabBytes - kFrameBytes);
    uint32_t *const fs = fr + 3 * kChan;  // scalars
    __syncwarp();
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t ch = lane + 32 * k;
        fr[ch] = c.off[k];
        fr[kChan + ch] = c.len[k];
        fr[2 * kChan + ch] = exs[k] | (((c.opens >> k) & 1u) << 31);  // (strips 16 bits, runs 14 bits)
    }
    if (lane == 0) {
        fs[0] = tot;
        fs[1] = c.fed_size;
        fs[2] = static_cast<uint32_t>(plan);
        fs[3] = static_cast<uint32_t>(plan >> 32);
        fs[4] = n_pieces;
        fs[5] = c.overrun;
        fs[6] = c.n_malformed;
        fs[7] = c.fed_start;
        fs[8] = fs[9] = fs[10] = fs[11] = fs[12] = 0;  // clusters, ADC bytes, seeds, entries, non-zero entries so far
        fs[13] = c.fo0;
        fs[14] = static_cast<uint32_t>(c.t_prev);  // (tracing)
        fs[15] = static_cast<uint32_t>(static_cast<unsigned long long>(c.t_prev) >> 32);
    }
    for (uint32_t i = 0;; ++i) {
        __syncwarp();  // every lane is done with the previous piece; the frame is written
        if (i >= fs[4]) break;
        const unsigned long long pl = fs[2] | (static_cast<unsigned long long>(fs[3]) << 32);
        const uint32_t b0 = i ? static_cast<uint32_t>(pl >> (8u * (i - 1u))) & 0xffu : 0u;
        const uint32_t b1 = static_cast<uint32_t>(pl >> (8u * i)) & 0xffu;
        const uint32_t fed_size = fs[1], over = fs[5];
        const uint32_t off_b0 = b0 < static_cast<uint32_t>(kChan) ? fr[b0] : fed_size + 2u;
        const uint32_t off_b1 = b1 < static_cast<uint32_t>(kChan) ? fr[b1] : fed_size + 2u;
        const uint32_t ex0 = (b0 < static_cast<uint32_t>(kChan) ? fr[2 * kChan + b0] : fs[0]) & 0x7fffffffu;
        const uint32_t ex1 = (b1 < static_cast<uint32_t>(kChan) ? fr[2 * kChan + b1] : fs[0]) & 0x7fffffffu;
        const uint32_t g_lo = (off_b0 - 2u) & ~15u;
        const uint32_t g_hi = over || b1 >= static_cast<uint32_t>(kChan) ? fed_size : (off_b1 - 2u + 15u) & ~15u;
        FedCtx pc;
        pc.ev = ticket - f * p.n_events;
        pc.f = f;
        pc.fo0 = fs[13];
        pc.fed_start = fs[7];
        pc.overrun = over;
        pc.n_malformed = fs[6];
        pc.opens = 0;
        pc.t_prev = kTrace ? static_cast<long long>(fs[14] | (static_cast<unsigned long long>(fs[15]) << 32)) : 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const uint32_t ch = lane + 32 * k;
            const bool in = ch >= b0 && ch < b1;
            const uint32_t xk = fr[2 * kChan + ch];
            pc.off[k] = in ? fr[ch] - g_lo : 0u;
            pc.len[k] = in ? fr[kChan + ch] : 0u;
            pc.ebase[k] = in ? (xk & 0xffffu) - (ex0 & 0xffffu) : 0u;
            pc.opens |= (xk >> 31) << k;
            if (in) ktab[ch] = pc.off[k] - pc.ebase[k] - 2u * (((xk >> 16) & 0x3fffu) - (ex0 >> 16));
        }
        pc.fed_size = g_hi - g_lo;
        pc.P = (ex1 & 0xffffu) - (ex0 & 0xffffu);
        pc.ch_lo = b0;
        pc.ch_hi = b1;
        pc.last = i + 1u == fs[4];
        pc.cl_base = fs[8];
        pc.adc_base = fs[9];
        pc.seed_base = fs[10];
        pc.ent_base = fs[11];
        pc.nz_base = fs[12];
        if (i > 0 && g_hi > g_lo) {
            __syncwarp();
            if (lane == 0) {
                fence_proxy_async();
                mbar_expect_tx(mbar, g_hi - g_lo);
                bulk_g2s(slot, p.ev[pc.ev].raw + pc.fed_start + g_lo, g_hi - g_lo, mbar, policy_evict_first());
            }
            mbar_wait(mbar, mbar_phase);
            mbar_phase ^= 1u;
        }
        __syncwarp();
        if (!fed_lists<true, true, kTrace>(p, slot, slot, pc, lane, next_ticket)) return false;
        if (lane == 0) {
            fs[8] = pc.cl_base;
            fs[9] = pc.adc_base;
            fs[10] = pc.seed_base;
            fs[11] = pc.ent_base;
            fs[12] = pc.nz_base;
            fs[14] = static_cast<uint32_t>(pc.t_prev);
            fs[15] = static_cast<uint32_t>(static_cast<unsigned long long>(pc.t_prev) >> 32);
        }
    }
    return true;
}

// ------------------------------------------------------------------------------ a7, second half, in the same launch
// The ordered move of one (event, FED) by a warp of sst_event_kernel that found the FED tickets
// used up (launches with plain outputs: cluster arrays, seeds, S/N).  Two round trips to memory per
// FED instead of one per array and loop: (1) the FED's own state word (acquire: what its warp staged
// is read afterwards), the words of its predecessors (their sum is the FED's place in the event's
// arrays) and its start offset, all in flight together; (2) ONE set of TMA bulk copies that brings
// the FED's staged records, ADC offsets and cluster ADCs into the warp's shared-memory slot, which
// is free by now.  The lanes then read shared memory and stream the arrays out.
__device__ __forceinline__ unsigned long long ld_state(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_state_acquire(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
constexpr uint32_t kMoveAdc = 1024;  // cluster ADC bytes per bulk copy (+ 32 for the alignment of both ends)

__device__ __forceinline__ void move_fed(const KParams &p, unsigned long long *mbar, uint8_t *slot, uint32_t &mbar_phase,
                                         const uint32_t ev, const uint32_t f, const int lane) {
    const EventDesc &E = p.ev[ev];
    const sst_output &o = E.out;
    const unsigned long long *const st = p.fed_state + static_cast<size_t>(ev) * p.n_feds;
    const uint32_t fed_start = __ldg(E.fed_offsets + f);
    const uint32_t epoch = warp_epoch(slot);
    // ---- round trip 1: state words.  clusters | ADC bytes << 32 ; seeds | malformed << 32 | overrun << 52
    unsigned long long own, accA, accB;
    for (uint32_t tries = 0;; ++tries) {
        own = ld_state_acquire(st + f);
        // (after a miss: wait for the FED's own word alone -- in FED-major order it is the last to appear)
        while (tries && static_cast<uint32_t>(own >> kShEpoch) != epoch) {
            __nanosleep(400);
            own = ld_state_acquire(st + f);
        }
        bool ok = static_cast<uint32_t>(own >> kShEpoch) == epoch;
        accA = accB = 0;
        constexpr int kW = 14;  // words per lane in flight (448 FEDs per pass)
#pragma unroll 1
        for (uint32_t j0 = lane; j0 < f; j0 += 32 * kW) {
            unsigned long long v[kW];
#pragma unroll
            for (int k = 0; k < kW; ++k) {
                const uint32_t j = j0 + 32 * k;
                v[k] = static_cast<unsigned long long>(epoch) << kShEpoch;
                if (j < f) v[k] = ld_state(st + j);
            }
#pragma unroll
            for (int k = 0; k < kW; ++k) {
                ok = ok && static_cast<uint32_t>(v[k] >> kShEpoch) == epoch;
                accA += (v[k] & 0x3fffull) | (((v[k] >> kShAdc) & 0x7fffull) << 32);
                accB += ((v[k] >> kShSeed) & 0x7fffull) | (((v[k] >> kShMalf) & 0x7full) << 32) | (((v[k] >> kShOver) & 1ull) << 52);
            }
        }
        if (__all_sync(kFull, ok)) break;
        __nanosleep(400);  // some earlier FED of the event is still being worked on
    }
    accA = warp_sum64(accA);
    accB = warp_sum64(accB);
    const uint32_t fed_cl = static_cast<uint32_t>(own & 0x3fffull), fed_adc = static_cast<uint32_t>((own >> kShAdc) & 0x7fffull),
                   fed_seed = static_cast<uint32_t>((own >> kShSeed) & 0x7fffull),
                   fed_malf = static_cast<uint32_t>((own >> kShMalf) & 0x7full), fed_over = static_cast<uint32_t>((own >> kShOver) & 1ull);
    const uint32_t b_cl = static_cast<uint32_t>(accA), b_adc = static_cast<uint32_t>(accA >> 32);
    const uint32_t b_seed = static_cast<uint32_t>(accB), b_malf = static_cast<uint32_t>(accB >> 32) & 0xfffffu,
                   b_over = static_cast<uint32_t>(accB >> 52);
    // where the FED's warp staged it (a FED with bad offsets staged nothing: its counts are zero)
    const size_t sb = static_cast<size_t>(ev) * p.s_cl_stride + fed_start / 2u + f;
    const size_t ab = static_cast<size_t>(ev) * p.g_ents + fed_start;
    const unsigned long long pol_first = policy_evict_first();
    const bool all_fit = b_cl + fed_cl <= o.cap_clusters && b_adc + fed_adc <= o.cap_adc;

    // ---- round trip 2: the staged FED into the slot: [records C x 16 | ADC offsets (C + 8) x 4 | cluster ADCs]
    const uint32_t C = p.move_chunk;
    const uint4 *const sm_rec = reinterpret_cast<const uint4 *>(slot);
    const uint32_t *const sm_off = reinterpret_cast<const uint32_t *>(slot + 16u * C);
    const uint8_t *const sm_adc = slot + 16u * C + 4u * (C + 8u);
    uint32_t off_sh = 0, adc_sh = 0;  // where the first wanted element sits in the (16-byte aligned) windows copied
    auto fetch = [&](const uint32_t k0, const uint32_t a0, const bool want_adc) {
        // clusters [k0, k0 + n) and/or ADC bytes [a0, a0 + m); windows rounded out to 16 bytes
        const uint32_t n = k0 < fed_cl ? min(C, fed_cl - k0) : 0u;
        const uint32_t m = want_adc && a0 < fed_adc ? min(kMoveAdc, fed_adc - a0) : 0u;
        const size_t o_lo = (sb + k0) & ~static_cast<size_t>(3), o_hi = (sb + k0 + n + 3u) & ~static_cast<size_t>(3);
        const size_t a_lo = (ab + a0) & ~static_cast<size_t>(15), a_hi = (ab + a0 + m + 15u) & ~static_cast<size_t>(15);
        if (n) off_sh = static_cast<uint32_t>(sb + k0 - o_lo);
        if (m) adc_sh = static_cast<uint32_t>(ab + a0 - a_lo);
        __syncwarp();  // every lane is done with what the slot held
        if (lane == 0) {
            // earlier generic-proxy accesses to the slot before the async writes; and, on the reader's
            // side too, the staging in global memory (seen through the acquire of the state words)
            // before the async reads
            asm volatile("fence.proxy.async;" ::: "memory");
            const uint32_t bytes = n * 16u + (n ? static_cast<uint32_t>(o_hi - o_lo) * 4u : 0u) + (m ? static_cast<uint32_t>(a_hi - a_lo) : 0u);
            mbar_expect_tx(mbar, bytes);
            if (n) {
                bulk_g2s(slot, p.s_rec + sb + k0, n * 16u, mbar, pol_first);
                bulk_g2s(slot + 16u * C, p.s_off + o_lo, static_cast<uint32_t>(o_hi - o_lo) * 4u, mbar, pol_first);
            }
            if (m) bulk_g2s(slot + 16u * C + 4u * (C + 8u), p.s_adc + a_lo, static_cast<uint32_t>(a_hi - a_lo), mbar, pol_first);
        }
        mbar_wait(mbar, mbar_phase);
        mbar_phase ^= 1u;
    };
    uint32_t lim = 0;  // ADC bytes of this FED that belong to clusters that fit
    if (fed_cl) {
        fetch(0, 0, true);
#pragma unroll 1
        for (uint32_t k0 = 0;;) {
            const uint32_t n = min(C, fed_cl - k0);
#pragma unroll 2
            for (uint32_t i = lane; i < n; i += 32) {
                const uint4 r = sm_rec[i];
                const uint32_t off = sm_off[off_sh + i];
                const uint32_t wd = r.y >> 16;
                const uint32_t k_cl = b_cl + k0 + i, k_adc = b_adc + off;
                if (all_fit || (k_cl < o.cap_clusters && k_adc + wd <= o.cap_adc)) {
                    st_stream(o.cl_module + k_cl, r.x, pol_first);
                    st_stream(o.cl_first + k_cl, r.y & 0xffffu, pol_first);
                    st_stream(o.cl_width + k_cl, wd, pol_first);
                    st_stream(o.cl_charge + k_cl, static_cast<int32_t>(r.z), pol_first);
                    st_stream(o.cl_bary + k_cl, __uint_as_float(r.w), pol_first);
                    st_stream(o.cl_adc_off + k_cl, k_adc, pol_first);
                    if (o.cl_snr) o.cl_snr[k_cl] = __ldcg(p.s_snr + sb + k0 + i);
                    lim = max(lim, off + wd);
                } else {
                    // the first cluster that does not fit reports how many were written
                    const bool prev_fits = k_cl == 0 || (k_cl - 1 < o.cap_clusters && k_adc <= o.cap_adc);
                    if (prev_fits) *o.n_clusters = k_cl;
                }
            }
            k0 += n;
            if (k0 >= fed_cl) break;
            fetch(k0, 0, false);
        }
        lim = all_fit ? fed_adc : __reduce_max_sync(kFull, lim);
        // cluster ADCs: aligned 32-bit words of the output from two aligned words of the slot
#pragma unroll 1
        for (uint32_t a0 = 0; a0 < lim;) {
            const uint32_t m = min(kMoveAdc, lim - a0);
            uint8_t *const D = o.cl_adc + b_adc + a0;
            const uint32_t head = min(m, (4u - (static_cast<uint32_t>(reinterpret_cast<uintptr_t>(D)) & 3u)) & 3u);
            const uint32_t nw = (m - head) >> 2, tail = (m - head) & 3u;
            if (static_cast<uint32_t>(lane) < head) st_stream(D + lane, sm_adc[adc_sh + lane], pol_first);
            if (static_cast<uint32_t>(lane) < tail) st_stream(D + head + 4u * nw + lane, sm_adc[adc_sh + head + 4u * nw + lane], pol_first);
#pragma unroll 2
            for (uint32_t w = lane; w < nw; w += 32) {
                const uint32_t s = adc_sh + head + 4u * w;
                const uint32_t *q = reinterpret_cast<const uint32_t *>(sm_adc + (s & ~3u));
                st_stream(reinterpret_cast<uint32_t *>(D + head) + w, __funnelshift_r(q[0], q[1], 8u * (s & 3u)), pol_first);
            }
            a0 += m;
            if (a0 < lim) fetch(fed_cl, a0, true);
        }
    }
    if (o.seed_idx) {
#pragma unroll 1
        for (uint32_t i = lane; i < fed_seed; i += 32)
            if (b_seed + i < o.cap_seeds) o.seed_idx[b_seed + i] = f * kFedStrips + __ldcg(p.s_seed + ab + i);
    }
    if (f == p.n_feds - 1 && lane == 0) {  // event totals = prefix of the last FED + its own
        const uint32_t t_cl = b_cl + fed_cl, t_adc = b_adc + fed_adc, n_mal = b_malf + fed_malf, n_over = b_over + fed_over;
        uint32_t flags = 0;
        if (t_cl > o.cap_clusters) flags |= SST_FLAG_CLUSTER_CAP;
        if (t_adc > o.cap_adc) flags |= SST_FLAG_ADC_CAP;
        if (n_mal) flags |= SST_FLAG_MALFORMED;
        if (n_over) flags |= SST_FLAG_OVERRUN;
        if (!(flags & (SST_FLAG_CLUSTER_CAP | SST_FLAG_ADC_CAP))) *o.n_clusters = t_cl;
        o.dev_status[SST_ST_FLAGS] = flags;
        o.dev_status[SST_ST_N_MALFORMED] = n_mal;
        o.dev_status[SST_ST_N_CLUSTERS] = t_cl;
        o.dev_status[SST_ST_N_ADC] = t_adc;
        o.dev_status[SST_ST_N_OVERRUN] = n_over;
        o.dev_status[SST_ST_N_SEEDS] = b_seed + fed_seed;
        o.dev_status[SST_ST_N_PRESENT] = 0;
        o.dev_status[7] = 0;
    }
}

// Tickets total .. 2 * total - 1 are the (event, FED) pairs again, in the same FED-major order.  A
// warp that finds the FED tickets used up moves staged FEDs while the last FEDs are still being
// worked on by others; a pair is moved once it and all its predecessors of the event carry this
// launch's epoch.  Every warp of the grid is resident (the grid never exceeds the resident
// capacity) and every FED ticket has been drawn by a running warp before the first move ticket is,
// so a wait always ends.
template <bool kTrace>
__device__ __forceinline__ void move_phase(const KParams &p, unsigned long long *mbar, uint8_t *slot, uint32_t &mbar_phase,
                                           uint32_t ticket, const uint32_t total, const int lane) {
    while (ticket < 2u * total) {
        const uint32_t t = ticket - total;
        uint32_t next_ticket = 0;
        if (lane == 0) next_ticket = static_cast<uint32_t>(atomicAdd(p.ticket, 1ull));
        const uint32_t f = t / p.n_events;
        const long long t0 = kTrace ? clock64() : 0;
        move_fed(p, mbar, slot, mbar_phase, t - f * p.n_events, f, lane);
        if (kTrace && lane == 0) {
            atomicAdd(p.trace + kTrMoveCycles, static_cast<unsigned long long>(clock64() - t0));
            atomicAdd(p.trace + kTrMoved, 1ull);
        }
        ticket = __shfl_sync(kFull, next_ticket, 0);
    }
}

// ------------------------------------------------------------------------------ the kernel
// Every warp works alone: it draws (event, FED) tickets until the launch's work is used up and
// never meets a block-wide barrier.  A CTA is just 1..kWarpsPerCta such warps sharing the SM's
// shared memory (one driver reserve per CTA instead of one per warp).
template <bool kPieces, bool kTrace>
__global__ void __launch_bounds__(32 * kWarpsPerCta, kMinCtas) sst_event_kernel(const __grid_constant__ KParams p) {
    extern __shared__ __align__(128) uint8_t smem_raw[];
    const int lane = threadIdx.x & 31;
    uint8_t *const mine = smem_raw + static_cast<size_t>(threadIdx.x >> 5) * (kWarpHdr + p.slot_bytes + kTailPad);
    unsigned long long *const mbar = reinterpret_cast<unsigned long long *>(mine);
    uint8_t *const slot = mine + kWarpHdr;
    if (lane == 0) {
        mbar_init(mbar, 1);
        fence_proxy_async();
        *reinterpret_cast<uint32_t *>(mine + 8) = launch_epoch(p);
    }
    __syncwarp();
    const uint32_t total = p.n_events * p.n_feds;
    auto wall_ns = [] {  // tracing: the launch's timeline on the GPU's nanosecond clock
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        return t;
    };
    if (kTrace && lane == 0) atomicMin(p.trace + kTrStart, wall_ns());
    uint32_t mbar_phase = 0;
    uint32_t ticket = 0;
    if (lane == 0) ticket = static_cast<uint32_t>(atomicAdd(p.ticket, 1ull));
    ticket = __shfl_sync(kFull, ticket, 0);
    while (ticket < total) {
        uint32_t next_ticket = 0;
        for (bool slow = false; !process_fed<kPieces, kTrace>(p, mbar, slot, ticket, lane, slow, mbar_phase, next_ticket); slow = true) {
        }  // (a FED whose cluster list outgrows the slot is redone through the global scratch)
        ticket = __shfl_sync(kFull, next_ticket, 0);
    }
    // The ordered move, in the same launch (plain outputs only): tickets total .. 2 * total - 1 are
    // the (event, FED) pairs again, in the same FED-major order.  A warp that finds the FED tickets
    // used up moves staged FEDs while the last FEDs are still being worked on by others; a pair is
    // moved once it and all its predecessors of the event carry this launch's epoch.  Every warp of
    // the grid is resident (the grid never exceeds the resident capacity) and every FED ticket has
    // been drawn by a running warp before the first move ticket is, so the wait always ends.
    if (kTrace && lane == 0) {
        const unsigned long long t = wall_ns();
        atomicMin(p.trace + kTrFirstOut, t);
        atomicMax(p.trace + kTrLastOut, t);
    }
    if (p.fused_move) move_phase<kTrace>(p, mbar, slot, mbar_phase, ticket, total, lane);
    if (kTrace && lane == 0) atomicMax(p.trace + kTrEnd, wall_ns());
    // The last warp of the launch to get here leaves the stream's header ready for the next launch:
    // ticket counter and warp count at zero, one launch more -- and when the epoch starts over with
    // that, the TAG of every FED state word cleared (tag 0 is no launch's epoch), so that a word of
    // this round of epochs is never taken for one of the next.  The counts stay: sst_emit_kernel,
    // when it runs behind this launch, still reads them (it ignores the tags).  (The launch's
    // parameters hold nothing that changes from launch to launch.)
    // The fences order this warp's earlier writes before its count, and the header writes below
    // after the counts of all the others.
    uint32_t left = 0;
    if (lane == 0) {
        __threadfence();
        left = static_cast<uint32_t>(atomicAdd(p.ticket + 1, 1ull)) + 1u == gridDim.x * (blockDim.x >> 5);
        __threadfence();
    }
    if (__shfl_sync(kFull, left, 0)) {
        const unsigned long long n = p.ticket[2] + 1ull == kEpochs ? 0ull : p.ticket[2] + 1ull;
        if (n == 0) {
#pragma unroll 1
            for (uint32_t i = lane; i < p.state_words; i += 32) p.fed_state[i] &= (1ull << kShEpoch) - 1ull;
        }
        __syncwarp();
        if (lane == 0) {
            p.ticket[0] = 0ull;
            p.ticket[1] = 0ull;
            p.ticket[2] = n;
        }
    }
}

// ------------------------------------------------------------------------------ a7, second half
// One warp per (event, FED), behind sst_event_kernel on the same stream: sums the state words of
// the FED's predecessors (exclusive prefix of clusters, ADC bytes, seeds), then moves the staged
// records, cluster ADCs and seeds of the FED to their final place.  Output capacity and the event
// totals are handled here.
// kExtras: some event of the launch wants hit coordinates or the compact SoA (an instantiation of
// its own, so that the plain move keeps its registers for loads in flight).
template <bool kPacked, bool kExtras>
__global__ void __launch_bounds__(128, kEmitCtas) sst_emit_kernel(const __grid_constant__ KParams p) {
    const int lane = threadIdx.x & 31;
    const uint32_t t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= p.n_events * p.n_feds) return;
    const uint32_t ev = t / p.n_feds, f = t - ev * p.n_feds;
    const EventDesc &E = p.ev[ev];
    sst_output o = E.out;
    constexpr bool packed = kPacked;  // every event of a launch is, or none
    // programmatic dependent launch: this grid may become resident while sst_event_kernel drains;
    // nothing of that kernel is read before it has completed
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const unsigned long long *const st = p.fed_state + static_cast<size_t>(ev) * p.n_feds;
    const unsigned long long own = st[f];
    const uint32_t fed_cl = static_cast<uint32_t>(own & 0x3fffull), fed_adc = static_cast<uint32_t>((own >> kShAdc) & 0x7fffull),
                   fed_seed = static_cast<uint32_t>((own >> kShSeed) & 0x7fffull),
                   fed_malf = static_cast<uint32_t>((own >> kShMalf) & 0x7full), fed_over = static_cast<uint32_t>((own >> kShOver) & 1ull);
    // clusters | ADC bytes << 32 ; seeds | malformed << 32 (20 bits) | overrun << 52 (n_feds <= 4096)
    unsigned long long accA = 0, accB = 0, totA = 0;
    const uint32_t jend = packed ? p.n_feds : f;  // the packed layout needs the event's totals too
#pragma unroll 8
    for (uint32_t j = lane; j < jend; j += 32) {
        const unsigned long long v = st[j];
        const unsigned long long a = (v & 0x3fffull) | (((v >> kShAdc) & 0x7fffull) << 32);
        totA += a;
        if (j < f) {
            accA += a;
            accB += ((v >> kShSeed) & 0x7fffull) | (((v >> kShMalf) & 0x7full) << 32) | (((v >> kShOver) & 1ull) << 52);
        }
    }
    accA = warp_sum64(accA);
    accB = warp_sum64(accB);
    if (packed) {
        // one block per event: {dev_status[8], n_clusters, pad to 64 B}, then the arrays back to
        // back with K = min(clusters found, cap_clusters) elements each: module, charge, bary,
        // adc_off (4 B), first, width (2 B), and the cluster ADCs -- one download per event
        const size_t K = min(static_cast<uint32_t>(warp_sum64(totA)), o.cap_clusters);
        uint8_t *b = E.packed;
        o.dev_status = reinterpret_cast<uint32_t *>(b);
        o.n_clusters = reinterpret_cast<uint32_t *>(b + 32);
        o.cl_module = reinterpret_cast<uint32_t *>(b + 64);
        o.cl_charge = reinterpret_cast<int32_t *>(b + 64 + 4 * K);
        o.cl_bary = reinterpret_cast<float *>(b + 64 + 8 * K);
        o.cl_adc_off = reinterpret_cast<uint32_t *>(b + 64 + 12 * K);
        o.cl_first = reinterpret_cast<uint16_t *>(b + 64 + 16 * K);
        o.cl_width = reinterpret_cast<uint16_t *>(b + 64 + 18 * K);
        o.cl_adc = b + 64 + 20 * K;
    }
    const uint32_t b_cl = static_cast<uint32_t>(accA), b_adc = static_cast<uint32_t>(accA >> 32);
    const uint32_t b_seed = static_cast<uint32_t>(accB), b_malf = static_cast<uint32_t>(accB >> 32) & 0xfffffu,
                   b_over = static_cast<uint32_t>(accB >> 52);
    // where sst_event_kernel staged this FED (a FED with bad offsets staged nothing: its counts
    // are zero and the addresses below are never used)
    const uint32_t fed_start = E.fed_offsets[f];
    const size_t sb = static_cast<size_t>(ev) * p.s_cl_stride + fed_start / 2u + f;
    const size_t ab = static_cast<size_t>(ev) * p.g_ents + fed_start;
    const unsigned long long pol_first = policy_evict_first();

    const bool all_fit = b_cl + fed_cl <= o.cap_clusters && b_adc + fed_adc <= o.cap_adc;
    uint32_t lim = 0;  // ADC bytes of this FED that belong to clusters that fit
    // the loop bodies first gather a few independent loads, then store: the kernel is a plain copy
    // and lives off loads in flight
    constexpr int kB = 4;
#pragma unroll 1
    for (uint32_t k0 = lane; k0 < fed_cl; k0 += 32 * kB) {
        uint4 r[kB];
        uint32_t off[kB];
        float snr[kB];
#pragma unroll
        for (int j = 0; j < kB; ++j) {
            const uint32_t k = k0 + 32 * j;
            if (k < fed_cl) {
                r[j] = p.s_rec[sb + k];
                off[j] = p.s_off[sb + k];
                if (o.cl_snr) snr[j] = p.s_snr[sb + k];
            }
        }
#pragma unroll
        for (int j = 0; j < kB; ++j) {
            const uint32_t k = k0 + 32 * j;
            if (k < fed_cl) {
                const uint32_t wd = r[j].y >> 16;
                const uint32_t k_cl = b_cl + k, k_adc = b_adc + off[j];
                if (all_fit || (k_cl < o.cap_clusters && k_adc + wd <= o.cap_adc)) {
                    st_stream(o.cl_module + k_cl, r[j].x, pol_first);
                    st_stream(o.cl_first + k_cl, r[j].y & 0xffffu, pol_first);
                    st_stream(o.cl_width + k_cl, wd, pol_first);
                    st_stream(o.cl_charge + k_cl, static_cast<int32_t>(r[j].z), pol_first);
                    st_stream(o.cl_bary + k_cl, __uint_as_float(r[j].w), pol_first);
                    st_stream(o.cl_adc_off + k_cl, k_adc, pol_first);
                    if (o.cl_snr) o.cl_snr[k_cl] = snr[j];
                    if (kExtras && o.hit_x) {  // clusters -> global hit coordinates (reading s23)
                        float hx = __int_as_float(0x7fc00000), hy = hx, hz = hx;
                        if (p.geom && r[j].x < p.n_geom) {
                            const float2 *gm = reinterpret_cast<const float2 *>(p.geom) + 3u * static_cast<size_t>(r[j].x);
                            const float2 g0 = __ldg(gm), g1 = __ldg(gm + 1), g2 = __ldg(gm + 2);  // {pitch, u0} {r, cos} {sin, z}
                            const float u = __fmaf_rn(g0.x, __uint_as_float(r[j].w), g0.y);
                            hx = __fmaf_rn(g1.x, g1.y, -__fmul_rn(u, g2.x));
                            hy = __fmaf_rn(g1.x, g2.x, __fmul_rn(u, g1.y));
                            hz = g2.y;
                        }
                        o.hit_x[k_cl] = hx;
                        o.hit_y[k_cl] = hy;
                        o.hit_z[k_cl] = hz;
                    }
                    lim = max(lim, off[j] + wd);
                } else {
                    // the first cluster that does not fit reports how many were written
                    const bool prev_fits = k_cl == 0 || (k_cl - 1 < o.cap_clusters && k_adc <= o.cap_adc);
                    if (prev_fits) *o.n_clusters = k_cl;
                }
            }
        }
    }
    lim = all_fit ? fed_adc : __reduce_max_sync(kFull, lim);
#pragma unroll 1
    for (uint32_t i0 = lane; i0 < lim; i0 += 32 * 8) {
        uint32_t v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if (i0 + 32 * j < lim) v[j] = p.s_adc[ab + i0 + 32 * j];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if (i0 + 32 * j < lim) st_stream(o.cl_adc + b_adc + i0 + 32 * j, v[j], pol_first);
    }
    if (o.seed_idx) {
#pragma unroll 1
        for (uint32_t i = lane; i < fed_seed; i += 32)
            if (b_seed + i < o.cap_seeds) o.seed_idx[b_seed + i] = f * kFedStrips + p.s_seed[ab + i];
    }
    // compact SoA, second half (on request): the FED's staged list goes to its place among the
    // event's recorded strips (exclusive prefix of the FEDs' non-zero entries), with the
    // calibration as it was uploaded gathered per entry
    uint32_t n_present = 0;
    if (kExtras && !packed && o.compact_strip) {
        const uint32_t *pr = p.fed_present + static_cast<size_t>(ev) * p.n_feds;
        uint32_t base = 0;
#pragma unroll 4
        for (uint32_t j = lane; j < f; j += 32) base += pr[j] & 0xffffu;
        base = __reduce_add_sync(kFull, base);
        const uint32_t own_p = pr[f], P = own_p >> 16;
        const uint32_t lt = (1u << lane) - 1u;
#pragma unroll 1
        for (uint32_t i0 = 0; i0 < P; i0 += 32) {
            const uint32_t i = i0 + lane;
            uint32_t a = 0, sid = 0;
            if (i < P) {
                a = p.s_cadc[ab + i];
                sid = p.s_csid[ab + i];
            }
            const uint32_t keep = __ballot_sync(kFull, a != 0);
            const uint32_t k = base + __popc(keep & lt);
            if (a != 0 && k < o.cap_compact) {
                const size_t g = static_cast<size_t>(f) * kFedStrips + sid;
                const float2 cv = __ldg(p.calib_orig + g);
                o.compact_strip[k] = static_cast<uint32_t>(g);
                o.compact_adc[k] = static_cast<uint8_t>(a);
                o.compact_noise[k] = cv.x;
                o.compact_gain[k] = cv.y;
                o.compact_bad[k] = __ldg(p.bad + g);
            }
            base += __popc(keep);
        }
        n_present = base;  // (of the last FED: the event's total)
    }
    if (f == p.n_feds - 1 && lane == 0) {  // event totals = prefix of the last FED + its own
        const uint32_t t_cl = b_cl + fed_cl, t_adc = b_adc + fed_adc, n_mal = b_malf + fed_malf, n_over = b_over + fed_over;
        uint32_t flags = 0;
        if (t_cl > o.cap_clusters) flags |= SST_FLAG_CLUSTER_CAP;
        if (t_adc > o.cap_adc) flags |= SST_FLAG_ADC_CAP;
        if (n_mal) flags |= SST_FLAG_MALFORMED;
        if (n_over) flags |= SST_FLAG_OVERRUN;
        if (n_present > o.cap_compact) flags |= SST_FLAG_COMPACT_CAP;
        if (!(flags & (SST_FLAG_CLUSTER_CAP | SST_FLAG_ADC_CAP))) *o.n_clusters = t_cl;
        o.dev_status[SST_ST_FLAGS] = flags;
        o.dev_status[SST_ST_N_MALFORMED] = n_mal;
        o.dev_status[SST_ST_N_CLUSTERS] = t_cl;
        o.dev_status[SST_ST_N_ADC] = t_adc;
        o.dev_status[SST_ST_N_OVERRUN] = n_over;
        o.dev_status[SST_ST_N_SEEDS] = b_seed + fed_seed;
        o.dev_status[SST_ST_N_PRESENT] = n_present;
        o.dev_status[7] = 0;
    }
}

}  // namespace

// ====================================================================================== host
struct sst_ctx {
    sst_config cfg{};
    cudaMemPool_t pool = nullptr;
    float2 *calib = nullptr;       // {noise (+inf at bad strips), gain}: what the kernels gather
    float2 *calib_orig = nullptr;  // {noise, gain} as uploaded
    uint8_t *bad = nullptr;        // bad flags as uploaded
    uint2 *chan_info = nullptr;
    float *geom = nullptr;         // module geometry for the hit conversion (sst_upload_geometry)
    uint32_t n_geom = 0;
    bool has_calib = false;
    std::atomic<int32_t> last_err{0};
    std::atomic<float> packed_ratio{0.0f};  // packed result bytes per raw byte seen by the last packed host call
    int sm_count = 0;
    int pieces = 1;            // > 1: the slot was sized for FEDs worked on in pieces (sst_event_kernel<true>)
    uint32_t whole_slot = 0;   // pieces > 1: slot that holds a whole large FED, for launches too small to fill
    int whole_warps_sm = 0;    //             the GPU (their latency is one FED's: pieces only add to it)
    int wpc = kWarpsPerCta;    // warps per CTA of a full launch
    int ctas_per_sm = 0;       // resident CTAs of wpc warps
    uint32_t slot_bytes = 0;   // shared-memory slot of one warp (one FED)
    uint32_t warp_stride = 0;  // mbarrier + slot + tail pad
    uint32_t smem_bytes = 0;   // kWarpsPerCta * warp_stride
    // per-stream scratch (launch header, FED states, slow-path lists), taken from the pool on a
    // stream's first launch and kept: stream order makes reuse safe, and every launch leaves the
    // header ready for the next
    // `captured`: a stream capture has recorded launches that point into `mem`; the block is then
    // never reallocated (a replay of that graph would use freed memory)
    struct Slot { cudaStream_t stream; uint8_t *mem; uint32_t cap_events; bool captured; };
    // cross-stream dependencies of the batched entry point: one event per stream, made on first use
    struct StreamEvent { cudaStream_t stream; cudaEvent_t ev; };
    std::vector<StreamEvent> stream_events;
    std::mutex slot_mu;
    std::vector<Slot> slots;
};

namespace {

inline bool cu_ok(sst_ctx *ctx, cudaError_t e) {
    if (e == cudaSuccess) return true;
    if (ctx) ctx->last_err.store(static_cast<int32_t>(e));
    return false;
}
#define SST_CU(call) \
    do { if (!cu_ok(ctx, (call))) return SST_ERR_CUDA; } while (0)

// the HOST entry points produce the cluster arrays, the dense SoA, the channel map and the seeds
bool no_device_only_outputs(const sst_output *o) { return !o->compact_strip && !o->hit_x && o->cap_compact == 0; }

// Gain correction without a division in the kernel (gain_apply): a factor c with
// min(254, floor(fma(adc, c, 0.5))) == min(254, floor(fl(fl(adc / gain) + 0.5))) -- the defining
// float32 form, reading s13 -- for EVERY adc in 1..255, searched among 1/gain and its
// float32 neighbours; -gain when none of them does (the kernel then divides for that strip).
// (double)adc * c is exact and so is the sum with 0.5 unless it is far below 1, where the floor is
// 0 either way: rounding it to float32 once is the fused multiply-add.
float gain_factor(const float g) {
    const float c0 = 1.0f / g;
    float cand[5] = {c0, std::nextafterf(c0, INFINITY), std::nextafterf(c0, 0.0f), 0.0f, 0.0f};
    cand[3] = std::nextafterf(cand[1], INFINITY);
    cand[4] = std::nextafterf(cand[2], 0.0f);
    for (const float c : cand) {
        if (!(c > 0.0f) || !std::isfinite(c)) continue;
        uint32_t diff = 0;
        for (int a = 1; a <= 255; ++a) {  // (no early exit: the loop vectorises)
            const float af = static_cast<float>(a);
            float u = af / g;
            u = u + 0.5f;
            const uint32_t ref = u >= 254.0f ? 254u : static_cast<uint32_t>(static_cast<int32_t>(u));
            const float v = static_cast<float>(static_cast<double>(af) * static_cast<double>(c) + 0.5);
            const uint32_t got = v >= 254.0f ? 254u : static_cast<uint32_t>(static_cast<int32_t>(v));
            diff |= ref ^ got;
        }
        if (diff == 0) return c;
    }
    return -g;
}

bool thresholds_ok(const sst_thresholds *t) {
    const float v[3] = {t->channel, t->seed, t->cluster};
    for (float x : v)
        if (!std::isfinite(x) || !(x > 0.0f)) return false;
    return true;
}

bool output_ok(const sst_output *o) {
    if (!(o && o->n_clusters && o->dev_status && o->cl_module && o->cl_first && o->cl_width && o->cl_charge &&
          o->cl_bary && o->cl_adc_off && o->cl_adc && !(o->seed_idx == nullptr && o->cap_seeds != 0)))
        return false;
    // the optional groups come complete or not at all
    const int nc = !!o->compact_strip + !!o->compact_adc + !!o->compact_noise + !!o->compact_gain + !!o->compact_bad;
    const int nh = !!o->hit_x + !!o->hit_y + !!o->hit_z;
    return (nc == 0 || nc == 5) && (nh == 0 || nh == 3) && !(nc == 0 && o->cap_compact != 0);
}

struct ScratchLayout {
    size_t ents, mwords, cl_slots, state_bytes, o_ticket, o_state, o_rec, o_mask, o_strip, o_adc, o_srec, o_soff, o_ssnr, o_present, o_csid, o_cadc,
        o_sadc, o_sseed, total;
};
ScratchLayout scratch_layout(const sst_ctx *ctx, size_t cap_events) {
    ScratchLayout L{};
    const uint32_t nf = ctx->cfg.n_feds;
    auto up = [](size_t b) { return (b + 255) & ~static_cast<size_t>(255); };
    L.ents = (static_cast<size_t>(ctx->cfg.max_raw_bytes) + 16ull * nf + 64 + 31) & ~static_cast<size_t>(31);
    L.mwords = L.ents / 32 + 4ull * nf + 16;
    // a cluster costs >= 2 raw bytes: one ADC byte and a separator (an inactive strip, or a run header)
    L.cl_slots = static_cast<size_t>(ctx->cfg.max_raw_bytes) / 2 + nf + 8;
    L.state_bytes = sizeof(unsigned long long) * nf * cap_events;
    L.o_ticket = 0;  // (+ 256: the 32 trace words)
    L.o_state = 512;
    // slow-path lists
    L.o_rec = L.o_state + up(L.state_bytes);
    L.o_mask = L.o_rec + up(4 * L.ents * cap_events);
    L.o_strip = L.o_mask + up(4 * 4 * L.mwords * cap_events);
    L.o_adc = L.o_strip + up(2 * L.ents * cap_events);
    // staging between the two kernels
    L.o_srec = L.o_adc + up(L.ents * cap_events);
    L.o_soff = L.o_srec + up(16 * L.cl_slots * cap_events);
    L.o_ssnr = L.o_soff + up(4 * L.cl_slots * cap_events);
    L.o_sadc = L.o_ssnr + up(4 * L.cl_slots * cap_events);
    L.o_sseed = L.o_sadc + up(L.ents * cap_events);
    L.o_present = L.o_sseed + up(2 * L.ents * cap_events);
    L.o_csid = L.o_present + up(L.state_bytes / 2);
    L.o_cadc = L.o_csid + up(2 * L.ents * cap_events);
    L.total = L.o_cadc + up(L.ents * cap_events);
    return L;
}

// Launches the two kernels for `n` (<= kMaxEv) events on `st`.  raw_limit[e] (NULL: the context's
// max_raw_bytes) is the number of readable bytes of raw[e].  The context's launch lock is held
// until both kernels are enqueued, so the ticket range a launch is given and the order in which
// the launches reach the stream always agree.
sst_status launch_events(sst_ctx *ctx, uint32_t n, const uint8_t *const *raw, const uint32_t *const *fed_offsets,
                         const sst_thresholds *thr, const sst_output *const *outs, cudaStream_t st,
                         uint8_t *const *packed = nullptr, const uint32_t *raw_limit = nullptr) {
    const uint32_t nf = ctx->cfg.n_feds;
    const uint32_t total = n * nf;
    // warps per CTA: full CTAs once the work fills the GPU, smaller ones to spread a small launch
    const uint32_t sms = static_cast<uint32_t>(ctx->sm_count);
    const uint32_t wfull = static_cast<uint32_t>(ctx->wpc);
    uint32_t wpc = std::min(wfull, total >= 16u * sms ? 8u : total >= 8u * sms ? 4u : total >= 4u * sms ? 2u : 1u);
    uint32_t capacity = static_cast<uint32_t>(ctx->sm_count * ctx->ctas_per_sm) * (wfull / wpc);
    uint32_t slot_bytes = ctx->slot_bytes;
    bool pieces = ctx->pieces > 1;
    // a launch that whole-FED slots can hold in one wave takes those: one warp per CTA, no pieces
    if (pieces && ctx->whole_slot && total <= sms * static_cast<uint32_t>(ctx->whole_warps_sm)) {
        pieces = false;
        slot_bytes = ctx->whole_slot;
        wpc = 1;
        capacity = sms * static_cast<uint32_t>(ctx->whole_warps_sm);
    }
    const uint32_t warp_stride = kWarpHdr + slot_bytes + kTailPad;
    const uint32_t grid = std::min((total + wpc - 1) / wpc, capacity);
    std::lock_guard<std::mutex> lock(ctx->slot_mu);
    sst_ctx::Slot *sl = nullptr;
    for (auto &s : ctx->slots)
        if (s.stream == st) sl = &s;
    if (!sl) {
        ctx->slots.push_back({st, nullptr, 0u, false});
        sl = &ctx->slots.back();
    }
    cudaStreamCaptureStatus capture = cudaStreamCaptureStatusNone;
    SST_CU(cudaStreamIsCapturing(st, &capture));
    const bool capturing = capture != cudaStreamCaptureStatusNone;
    if (sl->cap_events < n) {  // (re)allocate the stream's scratch for 1, 8, 16, 32 or kMaxEv events
        // not inside a capture (the allocation would become part of the graph) and not once a graph
        // holds the block's address: the stream must have seen a plain call at least this large before
        if (capturing || sl->captured) return SST_ERR_INVALID_ARG;
        if (sl->mem) SST_CU(cudaFreeAsync(sl->mem, st));
        sl->mem = nullptr;
        sl->cap_events = 0;
        const uint32_t want = n <= 1 ? 1u : n <= 8 ? 8u : n <= 16 ? 16u : n <= 32 ? 32u : static_cast<uint32_t>(kMaxEv);
        const ScratchLayout Ln = scratch_layout(ctx, want);
        uint8_t *mem = nullptr;
        SST_CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&mem), Ln.total, ctx->pool, st));
        if (!cu_ok(ctx, cudaMemsetAsync(mem, 0, Ln.o_rec, st))) {  // ticket counter and states
            cudaFreeAsync(mem, st);
            return SST_ERR_CUDA;
        }
        cudaMemsetAsync(mem + Ln.o_ticket + 256 + 8 * kTrStart, 0xff, 16, st);  // trace: the two minima
        sl->mem = mem;
        sl->cap_events = want;
    }
    if (capturing) sl->captured = true;
    uint8_t *const blk = sl->mem;
    const ScratchLayout L = scratch_layout(ctx, sl->cap_events);
    KParams kp{};
    kp.calib = ctx->calib;
    kp.chan_info = ctx->chan_info;
    kp.calib_orig = ctx->calib_orig;
    kp.bad = ctx->bad;
    kp.geom = ctx->geom;
    kp.n_geom = ctx->n_geom;
    kp.fed_present = reinterpret_cast<uint32_t *>(blk + L.o_present);
    kp.s_csid = reinterpret_cast<uint16_t *>(blk + L.o_csid);
    kp.s_cadc = blk + L.o_cadc;
    kp.ticket = reinterpret_cast<unsigned long long *>(blk + L.o_ticket);
    kp.state_words = static_cast<uint32_t>(sl->cap_events) * nf;
    kp.trace = reinterpret_cast<unsigned long long *>(blk + L.o_ticket + 256);
    kp.fed_state = reinterpret_cast<unsigned long long *>(blk + L.o_state);
    kp.g_rec = reinterpret_cast<uint32_t *>(blk + L.o_rec);
    kp.g_mask = reinterpret_cast<uint32_t *>(blk + L.o_mask);
    kp.g_strip = reinterpret_cast<uint16_t *>(blk + L.o_strip);
    kp.g_adc = blk + L.o_adc;
    kp.s_rec = reinterpret_cast<uint4 *>(blk + L.o_srec);
    kp.s_off = reinterpret_cast<uint32_t *>(blk + L.o_soff);
    kp.s_snr = reinterpret_cast<float *>(blk + L.o_ssnr);
    kp.s_adc = blk + L.o_sadc;
    kp.s_seed = reinterpret_cast<uint16_t *>(blk + L.o_sseed);
    kp.s_cl_stride = static_cast<uint32_t>(L.cl_slots);
    kp.g_ents = static_cast<uint32_t>(L.ents);
    kp.g_mwords = static_cast<uint32_t>(L.mwords);
    kp.tcl2 = static_cast<double>(thr->cluster) * static_cast<double>(thr->cluster);  // exact
    kp.t_ch = thr->channel;
    kp.t_seed = thr->seed;
    kp.max_raw_bytes = ctx->cfg.max_raw_bytes;
    kp.n_feds = nf;
    kp.n_events = n;
    kp.slot_bytes = slot_bytes;
    for (uint32_t e = 0; e < n; ++e) {
        kp.ev[e].raw = raw[e];
        kp.ev[e].fed_offsets = fed_offsets[e];
        kp.ev[e].out = *outs[e];
        kp.ev[e].packed = packed ? packed[e] : nullptr;
        kp.ev[e].raw_limit = raw_limit ? std::min(raw_limit[e], ctx->cfg.max_raw_bytes) : ctx->cfg.max_raw_bytes;
    }
    bool extras = false;
    for (uint32_t e = 0; e < n; ++e) extras = extras || outs[e]->hit_x || outs[e]->compact_strip;
    // plain outputs: sst_event_kernel moves the staged clusters itself (one launch); the packed
    // host block, hit coordinates and the compact SoA take sst_emit_kernel behind it
    const bool fused = !packed && !extras && ctx->cfg.move_mode == 0;
    kp.fused_move = fused ? 1u : 0u;
    kp.move_chunk = std::min(1024u, ((slot_bytes - (kMoveAdc + 32u) - 32u) / 20u) & ~31u);  // (slot_bytes >= 4096)
    const bool trace = ctx->cfg.trace != 0;
    if (pieces && trace) sst_event_kernel<true, true><<<grid, 32 * wpc, wpc * warp_stride, st>>>(kp);
    else if (pieces) sst_event_kernel<true, false><<<grid, 32 * wpc, wpc * warp_stride, st>>>(kp);
    else if (trace) sst_event_kernel<false, true><<<grid, 32 * wpc, wpc * warp_stride, st>>>(kp);
    else sst_event_kernel<false, false><<<grid, 32 * wpc, wpc * warp_stride, st>>>(kp);
    cudaError_t err = cudaGetLastError();
    if (err == cudaSuccess && !fused) {
        // the move is launched as a programmatic dependent of the event kernel: its CTAs are set up
        // while that kernel's last warps finish (the kernel itself waits for its completion)
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3((total + 3) / 4);
        lc.blockDim = dim3(128);
        lc.dynamicSmemBytes = 0;
        lc.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at;
        lc.numAttrs = 1;
        if (packed) err = cudaLaunchKernelEx(&lc, sst_emit_kernel<true, false>, kp);
        else if (extras) err = cudaLaunchKernelEx(&lc, sst_emit_kernel<false, true>, kp);
        else err = cudaLaunchKernelEx(&lc, sst_emit_kernel<false, false>, kp);  // (move_mode 1)
        if (err == cudaSuccess) err = cudaGetLastError();
    }
    if (err != cudaSuccess) {
        // (the header of a launch that did not happen is as the launch before left it; clearing the
        // ticket counter and the warp count again costs nothing)
        cu_ok(ctx, err);
        cudaMemsetAsync(blk, 0, 16, st);  // (ticket counter and warp count)
        return SST_ERR_CUDA;
    }
    return SST_OK;
}

}  // namespace

// ------------------------------------------------------ scratch of sst_unpack_cluster_noalloc
// The one block of scratch that is not taken from a pool: part of the library's device image, so
// every GPU that loads the kernels holds these 32 MiB until the process ends.  For callers that may
// not allocate once they run (include/sst.h).  HOST code must not use this name as a pointer: on the
// host it only stands for the symbol; noalloc_scratch() below asks the runtime for the device
// address, once per GPU.
static __device__ __align__(256) uint8_t sst_noalloc_scratch[SST_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
uint8_t *g_noalloc_ptr[kNoallocMaxDevices] = {};  // device address of sst_noalloc_scratch per GPU ordinal

// Device address of the static scratch on the context's GPU, which the caller has made current.
// The look-up (cudaGetSymbolAddress) runs on the first call per GPU and is remembered.
sst_status noalloc_scratch(sst_ctx *ctx, uint8_t **out) {
    const int dev = ctx->cfg.device;
    if (dev < 0 || dev >= kNoallocMaxDevices) return SST_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *ptr = nullptr;
        SST_CU(cudaGetSymbolAddress(&ptr, sst_noalloc_scratch));
        if (!ptr) return SST_ERR_CUDA;
        // also part of the set-up: have the runtime load the four kernels this entry point can launch
        // now, so that no later call is the first use of one (loading a kernel is the runtime's
        // business, but it is work a caller on a fixed budget wants behind it)
        cudaFuncAttributes fa;
        SST_CU(cudaFuncGetAttributes(&fa, sst_event_kernel<false, false>));
        SST_CU(cudaFuncGetAttributes(&fa, sst_event_kernel<true, false>));
        SST_CU(cudaFuncGetAttributes(&fa, sst_emit_kernel<false, false>));
        SST_CU(cudaFuncGetAttributes(&fa, sst_emit_kernel<false, true>));
        g_noalloc_ptr[dev] = static_cast<uint8_t *>(ptr);
    }
    *out = g_noalloc_ptr[dev];
    return SST_OK;
}

// One event on `st` with the static scratch at `blk` laid out as the pool scratch of one event is
// (scratch_layout(ctx, 1)); the launch itself is what launch_events does for n = 1.  Nothing here
// allocates.  The array holds what the last call -- of any context -- left: the launch header and
// the FED words are cleared first, so every call runs as a stream's very first launch (epoch 1).
sst_status launch_event_noalloc(sst_ctx *ctx, uint8_t *blk, const uint8_t *raw, const uint32_t *fed_offsets,
                                const sst_thresholds *thr, const sst_output *out, cudaStream_t st) {
    const ScratchLayout L = scratch_layout(ctx, 1);
    const uint32_t nf = ctx->cfg.n_feds;
    const uint32_t sms = static_cast<uint32_t>(ctx->sm_count);
    const uint32_t wfull = static_cast<uint32_t>(ctx->wpc);
    uint32_t wpc = std::min(wfull, nf >= 16u * sms ? 8u : nf >= 8u * sms ? 4u : nf >= 4u * sms ? 2u : 1u);
    uint32_t capacity = static_cast<uint32_t>(ctx->sm_count * ctx->ctas_per_sm) * (wfull / wpc);
    uint32_t slot_bytes = ctx->slot_bytes;
    bool pieces = ctx->pieces > 1;
    if (pieces && ctx->whole_slot && nf <= sms * static_cast<uint32_t>(ctx->whole_warps_sm)) {
        pieces = false;
        slot_bytes = ctx->whole_slot;
        wpc = 1;
        capacity = sms * static_cast<uint32_t>(ctx->whole_warps_sm);
    }
    const uint32_t warp_stride = kWarpHdr + slot_bytes + kTailPad;
    const uint32_t grid = std::min((nf + wpc - 1) / wpc, capacity);
    SST_CU(cudaMemsetAsync(blk, 0, L.o_rec, st));  // work counter, warp count, launch count; every FED word
    KParams kp{};
    kp.calib = ctx->calib;
    kp.chan_info = ctx->chan_info;
    kp.calib_orig = ctx->calib_orig;
    kp.bad = ctx->bad;
    kp.geom = ctx->geom;
    kp.n_geom = ctx->n_geom;
    kp.fed_present = reinterpret_cast<uint32_t *>(blk + L.o_present);
    kp.s_csid = reinterpret_cast<uint16_t *>(blk + L.o_csid);
    kp.s_cadc = blk + L.o_cadc;
    kp.ticket = reinterpret_cast<unsigned long long *>(blk + L.o_ticket);
    kp.state_words = nf;
    kp.trace = reinterpret_cast<unsigned long long *>(blk + L.o_ticket + 256);
    kp.fed_state = reinterpret_cast<unsigned long long *>(blk + L.o_state);
    kp.g_rec = reinterpret_cast<uint32_t *>(blk + L.o_rec);
    kp.g_mask = reinterpret_cast<uint32_t *>(blk + L.o_mask);
    kp.g_strip = reinterpret_cast<uint16_t *>(blk + L.o_strip);
    kp.g_adc = blk + L.o_adc;
    kp.s_rec = reinterpret_cast<uint4 *>(blk + L.o_srec);
    kp.s_off = reinterpret_cast<uint32_t *>(blk + L.o_soff);
    kp.s_snr = reinterpret_cast<float *>(blk + L.o_ssnr);
    kp.s_adc = blk + L.o_sadc;
    kp.s_seed = reinterpret_cast<uint16_t *>(blk + L.o_sseed);
    kp.s_cl_stride = static_cast<uint32_t>(L.cl_slots);
    kp.g_ents = static_cast<uint32_t>(L.ents);
    kp.g_mwords = static_cast<uint32_t>(L.mwords);
    kp.tcl2 = static_cast<double>(thr->cluster) * static_cast<double>(thr->cluster);
    kp.t_ch = thr->channel;
    kp.t_seed = thr->seed;
    kp.max_raw_bytes = ctx->cfg.max_raw_bytes;
    kp.n_feds = nf;
    kp.n_events = 1;
    kp.slot_bytes = slot_bytes;
    kp.ev[0].raw = raw;
    kp.ev[0].fed_offsets = fed_offsets;
    kp.ev[0].out = *out;
    kp.ev[0].packed = nullptr;
    kp.ev[0].raw_limit = ctx->cfg.max_raw_bytes;
    const bool extras = out->hit_x || out->compact_strip;
    const bool fused = !extras && ctx->cfg.move_mode == 0;
    kp.fused_move = fused ? 1u : 0u;
    kp.move_chunk = std::min(1024u, ((slot_bytes - (kMoveAdc + 32u) - 32u) / 20u) & ~31u);
    if (pieces) sst_event_kernel<true, false><<<grid, 32 * wpc, wpc * warp_stride, st>>>(kp);
    else sst_event_kernel<false, false><<<grid, 32 * wpc, wpc * warp_stride, st>>>(kp);
    cudaError_t err = cudaGetLastError();
    if (err == cudaSuccess && !fused) {
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3((nf + 3) / 4);
        lc.blockDim = dim3(128);
        lc.dynamicSmemBytes = 0;
        lc.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at;
        lc.numAttrs = 1;
        if (extras) err = cudaLaunchKernelEx(&lc, sst_emit_kernel<false, true>, kp);
        else err = cudaLaunchKernelEx(&lc, sst_emit_kernel<false, false>, kp);
        if (err == cudaSuccess) err = cudaGetLastError();
    }
    return cu_ok(ctx, err) ? SST_OK : SST_ERR_CUDA;
}

}  // namespace

extern "C" {

sst_status sst_create(const sst_config *cfg, sst_ctx **out_ctx) {
    if (out_ctx) *out_ctx = nullptr;
    if (!cfg || !out_ctx || cfg->n_feds == 0 || cfg->n_feds > kMaxFeds || cfg->max_raw_bytes == 0 ||
        cfg->move_mode > 1 || cfg->trace > 1)
        return SST_ERR_INVALID_ARG;
    sst_ctx *ctx = new (std::nothrow) sst_ctx();
    if (!ctx) return SST_ERR_INVALID_ARG;
    ctx->cfg = *cfg;
    if (ctx->cfg.max_events_in_flight == 0) ctx->cfg.max_events_in_flight = 8;
    auto fail = [&](sst_status s) {
        if (ctx->calib) cudaFree(ctx->calib);
        if (ctx->calib_orig) cudaFree(ctx->calib_orig);
        if (ctx->bad) cudaFree(ctx->bad);
        if (ctx->chan_info) cudaFree(ctx->chan_info);
        if (ctx->pool) cudaMemPoolDestroy(ctx->pool);
        delete ctx;
        return s;
    };
    if (cudaSetDevice(cfg->device) != cudaSuccess) return fail(SST_ERR_CUDA);
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = cfg->device;
    if (cudaMemPoolCreate(&ctx->pool, &props) != cudaSuccess) return fail(SST_ERR_CUDA);
    unsigned long long keep = ~0ull;  // never give memory back between events
    if (cudaMemPoolSetAttribute(ctx->pool, cudaMemPoolAttrReleaseThreshold, &keep) != cudaSuccess)
        return fail(SST_ERR_CUDA);
    const size_t n = static_cast<size_t>(cfg->n_feds) * kFedStrips;
    if (cudaMalloc(&ctx->calib, n * sizeof(float2)) != cudaSuccess) return fail(SST_ERR_CUDA);
    if (cudaMalloc(&ctx->calib_orig, n * sizeof(float2)) != cudaSuccess) return fail(SST_ERR_CUDA);
    if (cudaMalloc(&ctx->bad, n) != cudaSuccess) return fail(SST_ERR_CUDA);
    if (cudaMalloc(&ctx->chan_info, static_cast<size_t>(cfg->n_feds) * kChan * sizeof(uint2)) !=
        cudaSuccess)
        return fail(SST_ERR_CUDA);
    // Shared-memory slot of one warp, sized from the configuration's hints for the fast-path layout
    // of fed_lists (payload with the ADC list squeezed into it, the dense window's gap, strip ids,
    // masks, channel table); FEDs that do not fit take the slow path through the global scratch.
    // Warps per CTA and resident CTAs are then chosen for the most resident warps, and the slot is
    // grown to whatever the SM's shared memory leaves at that occupancy.
    cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, cfg->device);
    {
        const double m = static_cast<double>(cfg->max_raw_bytes) / cfg->n_feds;  // mean payload bound
        const uint32_t p_hint = cfg->fed_strips_hint ? std::min(cfg->fed_strips_hint, static_cast<uint32_t>(kFedStrips))
                                                     : static_cast<uint32_t>(0.5 * m) + 32u;
        const uint32_t r_hint = (static_cast<uint32_t>(std::min(1.15 * m + 64.0, 65536.0)) + 15u) & ~15u;
        int smem_optin = 0;
        cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, cfg->device);
        // The dynamic shared-memory limit is per-FUNCTION state shared by every context of the
        // process: it is set to the device maximum, never to this context's size, so contexts with
        // different slot sizes can be used side by side.
        if (cudaFuncSetAttribute(sst_event_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin) != cudaSuccess ||
            cudaFuncSetAttribute(sst_event_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin) != cudaSuccess ||
            cudaFuncSetAttribute(sst_event_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin) != cudaSuccess ||
            cudaFuncSetAttribute(sst_event_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin) != cudaSuccess)
            return fail(SST_ERR_CUDA);
        cudaFuncSetAttribute(sst_event_kernel<false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        cudaFuncSetAttribute(sst_event_kernel<true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        cudaFuncSetAttribute(sst_event_kernel<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        cudaFuncSetAttribute(sst_event_kernel<true, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        // A large FED may be worked on in K pieces (process_fed): the slot then holds the whole
        // payload while the channel table is built, and one piece's lists afterwards.  K = 1..4 is
        // tried, up to the first that keeps 20 warps resident per SM.
        int best_warps = 0;
        uint32_t need = 0, need_whole = 0;
        for (uint32_t K = 1; K <= 4; ++K) {
            const uint32_t pk = (p_hint + K - 1) / K + (K > 1 ? 64u : 0u);                      // strips of a piece
            const uint32_t rk = K > 1 ? ((r_hint / K + 256u + 15u) & ~15u) : r_hint;             // its payload bytes
            const uint32_t p16 = (pk + 15u) & ~15u;
            const uint32_t gap = rk >= p16 + 2048u ? 0u : p16 + 2048u - rk;
            uint32_t need_k = std::max(rk + gap + 2u * pk + 16u * (pk / 32u + 3u) + (K > 1 ? kFrameBytes : 0u), K > 1 ? r_hint : 0u) + kTabBytes + 32u;
            need_k = std::min(std::max((need_k + 15u) & ~15u, 4096u), (static_cast<uint32_t>(smem_optin) - kWarpHdr - kTailPad) & ~15u);
            const uint32_t stride = kWarpHdr + need_k + kTailPad;
            if (K == 1) need_whole = need_k;
            for (int wpc = kWarpsPerCta; wpc >= 1; wpc >>= 1) {
                int ctas = 0;
                if (static_cast<size_t>(wpc) * stride > static_cast<size_t>(smem_optin)) continue;
                if ((K > 1 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, sst_event_kernel<true, false>, 32 * wpc, static_cast<size_t>(wpc) * stride)
                           : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, sst_event_kernel<false, false>, 32 * wpc, static_cast<size_t>(wpc) * stride)) !=
                    cudaSuccess)
                    continue;
                if (ctas * wpc > best_warps) {
                    best_warps = ctas * wpc;
                    ctx->wpc = wpc;
                    ctx->ctas_per_sm = ctas;
                    ctx->pieces = static_cast<int>(K);
                    need = need_k;
                }
            }
            // pieces repeat the per-FED fixed work: they pay only while the SM is short of warps
            if (best_warps >= 20) break;
        }
        cudaGetLastError();
        if (best_warps < 1) return fail(SST_ERR_CUDA);
        auto set_slot = [&](uint32_t slot) {
            ctx->slot_bytes = slot;
            ctx->warp_stride = kWarpHdr + slot + kTailPad;
            ctx->smem_bytes = static_cast<uint32_t>(ctx->wpc) * ctx->warp_stride;
        };
        set_slot(need);
        // grow: first what the SM's shared memory divides into, then what the occupancy API offers
        int smem_sm = 0, smem_reserved = 0;
        cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, cfg->device);
        cudaDeviceGetAttribute(&smem_reserved, cudaDevAttrReservedSharedMemoryPerBlock, cfg->device);
        size_t api_avail = 0;
        if (ctx->pieces > 1) cudaOccupancyAvailableDynamicSMemPerBlock(&api_avail, sst_event_kernel<true, false>, ctx->ctas_per_sm, 32 * ctx->wpc);
        else cudaOccupancyAvailableDynamicSMemPerBlock(&api_avail, sst_event_kernel<false, false>, ctx->ctas_per_sm, 32 * ctx->wpc);
        const size_t tries[2] = {smem_sm > 0 ? static_cast<size_t>(smem_sm) / ctx->ctas_per_sm - smem_reserved : 0, api_avail};
        for (size_t avail : tries) {
            avail = std::min<size_t>(avail, static_cast<size_t>(smem_optin));
            if (avail <= ctx->smem_bytes) continue;
            const uint32_t slot = (static_cast<uint32_t>(avail / ctx->wpc) - kWarpHdr - kTailPad) & ~15u;
            if (slot <= ctx->slot_bytes) continue;
            const uint32_t keep = ctx->slot_bytes;
            set_slot(slot);
            int check = 0;
            if ((ctx->pieces > 1 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&check, sst_event_kernel<true, false>, 32 * ctx->wpc, ctx->smem_bytes)
                                 : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&check, sst_event_kernel<false, false>, 32 * ctx->wpc, ctx->smem_bytes)) == cudaSuccess &&
                check >= ctx->ctas_per_sm)
                break;
            set_slot(keep);  // the grown slot lost a CTA
        }
        if (ctx->pieces > 1) {
            int ctas = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, sst_event_kernel<false, false>, 32, kWarpHdr + need_whole + kTailPad) == cudaSuccess &&
                ctas > 0) {
                ctx->whole_slot = need_whole;
                ctx->whole_warps_sm = ctas;
            }
        }
        cudaGetLastError();
    }
    *out_ctx = ctx;
    return SST_OK;
}

sst_status sst_upload_calib(sst_ctx *ctx, const float *gain, const float *noise, const uint8_t *bad,
                            const uint32_t *chan_module) {
    if (!ctx || !gain || !noise || !bad || !chan_module) return SST_ERR_INVALID_ARG;
    const uint32_t nf = ctx->cfg.n_feds;
    const size_t n = static_cast<size_t>(nf) * kFedStrips, nch = static_cast<size_t>(nf) * kChan;
    for (size_t c = 1; c < nch; ++c) {
        if (chan_module[c] < chan_module[c - 1]) return SST_ERR_BAD_CALIB;
        if (c % kChan == 0 && chan_module[c] == chan_module[c - 1]) return SST_ERR_BAD_CALIB;
    }
    std::vector<float2> packed;
    try {
        packed.resize(n);
    } catch (...) {
        return SST_ERR_INVALID_ARG;
    }
    // {noise, gain factor} per strip, by all host cores: the factor search checks 255 ADC values
    // per candidate
    {
        std::atomic<bool> bad_calib{false};
        const unsigned nt = std::max(1u, std::min(32u, std::thread::hardware_concurrency()));
        auto work = [&](size_t g0, size_t g1) {
            for (size_t g = g0; g < g1; ++g) {
                if (bad[g]) {
                    // a bad strip is never active: noise = +inf fails every >= test; gain is never used
                    packed[g] = make_float2(INFINITY, 1.0f);
                } else {
                    if (!std::isfinite(gain[g]) || !(gain[g] > 0.0f) || !std::isfinite(noise[g]) || !(noise[g] > 0.0f)) {
                        bad_calib.store(true);
                        return;
                    }
                    packed[g] = make_float2(noise[g], gain_factor(gain[g]));
                }
            }
        };
        std::vector<std::thread> pool;
        const size_t per = (n + nt - 1) / nt;
        try {
            for (unsigned t = 1; t < nt; ++t)
                if (t * per < n) pool.emplace_back(work, t * per, std::min(n, (t + 1) * per));
        } catch (...) {  // no more threads: the rest is done here
        }
        const size_t started = pool.size();
        work(0, std::min(n, per));
        for (size_t t = started + 1; t < nt; ++t)
            if (t * per < n) work(t * per, std::min(n, (t + 1) * per));
        for (auto &th : pool) th.join();
        if (bad_calib.load()) return SST_ERR_BAD_CALIB;
    }
    SST_CU(cudaSetDevice(ctx->cfg.device));
    SST_CU(cudaMemcpy(ctx->calib, packed.data(), n * sizeof(float2), cudaMemcpyHostToDevice));
    // the values as given, for the compact SoA (PAPER.md:31 gathers the calibration into it)
    for (size_t g = 0; g < n; ++g) packed[g] = make_float2(noise[g], gain[g]);
    SST_CU(cudaMemcpy(ctx->calib_orig, packed.data(), n * sizeof(float2), cudaMemcpyHostToDevice));
    SST_CU(cudaMemcpy(ctx->bad, bad, n, cudaMemcpyHostToDevice));
    // module extent of every channel (modules are runs of equal ids inside one FED)
    std::vector<uint2> info(nch);
    for (size_t c0 = 0; c0 < nch;) {
        size_t c1 = c0 + 1;
        while (c1 < nch && c1 % kChan != 0 && chan_module[c1] == chan_module[c0]) ++c1;
        for (size_t c = c0; c < c1; ++c)
            info[c] = make_uint2(chan_module[c0], static_cast<uint32_t>(c0 % kChan) | (static_cast<uint32_t>((c1 - 1) % kChan + 1) << 8));
        c0 = c1;
    }
    SST_CU(cudaMemcpy(ctx->chan_info, info.data(), nch * sizeof(uint2), cudaMemcpyHostToDevice));
    SST_CU(cudaDeviceSynchronize());
    ctx->has_calib = true;
    return SST_OK;
}

sst_status sst_upload_geometry(sst_ctx *ctx, const float *geom, uint32_t n_modules) {
    if (!ctx || !geom || n_modules == 0) return SST_ERR_INVALID_ARG;
    for (size_t i = 0; i < static_cast<size_t>(n_modules) * 6; ++i)
        if (!std::isfinite(geom[i])) return SST_ERR_INVALID_ARG;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    SST_CU(cudaDeviceSynchronize());
    if (ctx->geom) cudaFree(ctx->geom);
    ctx->geom = nullptr;
    ctx->n_geom = 0;
    SST_CU(cudaMalloc(&ctx->geom, static_cast<size_t>(n_modules) * 6 * sizeof(float)));
    SST_CU(cudaMemcpy(ctx->geom, geom, static_cast<size_t>(n_modules) * 6 * sizeof(float), cudaMemcpyHostToDevice));
    ctx->n_geom = n_modules;
    return SST_OK;
}

sst_status sst_unpack_cluster(sst_ctx *ctx, const uint8_t *raw, const uint32_t *fed_offsets,
                              const sst_thresholds *thr, const sst_output *out, void *stream) {
    if (!ctx || !raw || !fed_offsets || !thr || !output_ok(out) || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    return launch_events(ctx, 1, &raw, &fed_offsets, thr, &out, static_cast<cudaStream_t>(stream));
}

// sst_unpack_cluster for callers that may not allocate (include/sst.h): the scratch is the static
// array above instead of a pool block.  The first call on a GPU also fetches the array's address.
sst_status sst_unpack_cluster_noalloc(sst_ctx *ctx, const uint8_t *raw, const uint32_t *fed_offsets,
                                      const sst_thresholds *thr, const sst_output *out, void *stream) {
    if (!ctx || !raw || !fed_offsets || !thr || !output_ok(out) || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    if (scratch_layout(ctx, 1).total > static_cast<size_t>(SST_NOALLOC_SCRATCH_BYTES)) return SST_ERR_TOO_LARGE;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    uint8_t *blk = nullptr;
    const sst_status s = noalloc_scratch(ctx, &blk);
    if (s != SST_OK) return s;
    return launch_event_noalloc(ctx, blk, raw, fed_offsets, thr, out, static_cast<cudaStream_t>(stream));
}

sst_status sst_unpack_cluster_batch(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                    const uint32_t *const *fed_offsets, const sst_thresholds *thr,
                                    const sst_output *outs, void *const *streams, uint32_t n_streams) {
    if (!ctx || !raw || !fed_offsets || !thr || !outs || !streams || n_streams == 0 || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    for (uint32_t e = 0; e < n_events; ++e)
        if (!raw[e] || !fed_offsets[e] || !output_ok(&outs[e])) return SST_ERR_INVALID_ARG;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    // Launch groups.  The events of all streams share one launch (two or more only beyond kMaxEv
    // events) so that the kernel walks them FED by FED (the FED's calibration slab is then read from
    // HBM once per launch, not once per event): stream s belongs to group s % G, the group's
    // launches run on its first stream, which
    // first waits for the other streams of the group (their uploads) and is waited for by them
    // afterwards, so every event's result is stream-ordered on its own stream as documented.
    const uint32_t ns = std::min(n_streams, n_events);
    const uint32_t G = std::min(ns, std::max(1u, (n_events + kMaxEv - 1) / kMaxEv));
    auto event_of = [&](cudaStream_t st, cudaEvent_t *out) -> bool {
        std::lock_guard<std::mutex> lock(ctx->slot_mu);
        for (auto &se : ctx->stream_events)
            if (se.stream == st) { *out = se.ev; return true; }
        cudaEvent_t ev = nullptr;
        if (!cu_ok(ctx, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming))) return false;
        ctx->stream_events.push_back({st, ev});
        *out = ev;
        return true;
    };
    for (uint32_t g = 0; g < G; ++g) {
        cudaStream_t lead = static_cast<cudaStream_t>(streams[g]);
        for (uint32_t s = g + G; s < ns; s += G) {  // the group's other streams: inputs ready
            cudaStream_t st = static_cast<cudaStream_t>(streams[s]);
            if (st == lead) continue;
            cudaEvent_t ev;
            if (!event_of(st, &ev)) return SST_ERR_CUDA;
            SST_CU(cudaEventRecord(ev, st));
            SST_CU(cudaStreamWaitEvent(lead, ev, 0));
        }
        const uint8_t *r[kMaxEv];
        const uint32_t *fo[kMaxEv];
        const sst_output *o[kMaxEv];
        uint32_t n = 0, left = 0;
        for (uint32_t e = 0; e < n_events; ++e)
            if ((e % n_streams) % G == g) ++left;
        for (uint32_t e = 0; e < n_events; ++e) {
            if ((e % n_streams) % G != g) continue;
            r[n] = raw[e];
            fo[n] = fed_offsets[e];
            o[n] = &outs[e];
            --left;
            if (++n == kMaxEv || left == 0) {
                const sst_status rc = launch_events(ctx, n, r, fo, thr, o, lead);
                if (rc != SST_OK) return rc;
                n = 0;
            }
        }
        bool others = false;
        for (uint32_t s = g + G; s < ns; s += G) others = others || static_cast<cudaStream_t>(streams[s]) != lead;
        if (others) {
            cudaEvent_t done;
            if (!event_of(lead, &done)) return SST_ERR_CUDA;
            SST_CU(cudaEventRecord(done, lead));
            for (uint32_t s = g + G; s < ns; s += G) {
                cudaStream_t st = static_cast<cudaStream_t>(streams[s]);
                if (st != lead) SST_CU(cudaStreamWaitEvent(st, done, 0));
            }
        }
    }
    return SST_OK;
}

sst_status sst_unpack_cluster_host(sst_ctx *ctx, const uint8_t *raw, uint32_t raw_bytes,
                                   const uint32_t *fed_offsets, const sst_thresholds *thr,
                                   const sst_output *out, void *stream) {
    if (!ctx || !raw || !fed_offsets || !thr || !output_ok(out) || !thresholds_ok(thr) || !no_device_only_outputs(out))
        return SST_ERR_INVALID_ARG;
    if (raw_bytes > ctx->cfg.max_raw_bytes) return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const uint32_t nf = ctx->cfg.n_feds;
    const size_t n = static_cast<size_t>(nf) * kFedStrips, nch = static_cast<size_t>(nf) * kChan;
    auto up = [](size_t b) { return (b + 255) & ~static_cast<size_t>(255); };
    // one pooled block, carved up
    const size_t o_raw = 0, o_fo = o_raw + up(ctx->cfg.max_raw_bytes), o_st = o_fo + up((nf + 1) * 4),
                 o_ncl = o_st + up(SST_ST_WORDS * 4), o_mod = o_ncl + 256,
                 o_first = o_mod + up(4ull * out->cap_clusters), o_width = o_first + up(2ull * out->cap_clusters),
                 o_charge = o_width + up(2ull * out->cap_clusters), o_bary = o_charge + up(4ull * out->cap_clusters),
                 o_aoff = o_bary + up(4ull * out->cap_clusters), o_snr = o_aoff + up(4ull * out->cap_clusters),
                 o_adc = o_snr + (out->cl_snr ? up(4ull * out->cap_clusters) : 0), o_dense = o_adc + up(out->cap_adc),
                 o_coff = o_dense + (out->strip_adc ? up(n) : 0), o_clen = o_coff + (out->chan_off ? up(4 * nch) : 0),
                 o_seed = o_clen + (out->chan_len ? up(2 * nch) : 0),
                 total = o_seed + (out->seed_idx ? up(4ull * out->cap_seeds) : 0);
    uint8_t *blk = nullptr;
    SST_CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&blk), total, ctx->pool, st));
    sst_status rc = SST_OK;
    auto CU = [&](cudaError_t e) { if (rc == SST_OK && !cu_ok(ctx, e)) rc = SST_ERR_CUDA; };
    CU(cudaMemcpyAsync(blk + o_raw, raw, raw_bytes, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(blk + o_fo, fed_offsets, (nf + 1) * 4, cudaMemcpyHostToDevice, st));
    sst_output d = *out;
    d.dev_status = reinterpret_cast<uint32_t *>(blk + o_st);
    d.n_clusters = reinterpret_cast<uint32_t *>(blk + o_ncl);
    d.cl_module = reinterpret_cast<uint32_t *>(blk + o_mod);
    d.cl_first = reinterpret_cast<uint16_t *>(blk + o_first);
    d.cl_width = reinterpret_cast<uint16_t *>(blk + o_width);
    d.cl_charge = reinterpret_cast<int32_t *>(blk + o_charge);
    d.cl_bary = reinterpret_cast<float *>(blk + o_bary);
    d.cl_adc_off = reinterpret_cast<uint32_t *>(blk + o_aoff);
    d.cl_snr = out->cl_snr ? reinterpret_cast<float *>(blk + o_snr) : nullptr;
    d.cl_adc = blk + o_adc;
    d.strip_adc = out->strip_adc ? blk + o_dense : nullptr;
    d.chan_off = out->chan_off ? reinterpret_cast<uint32_t *>(blk + o_coff) : nullptr;
    d.chan_len = out->chan_len ? reinterpret_cast<uint16_t *>(blk + o_clen) : nullptr;
    d.seed_idx = out->seed_idx ? reinterpret_cast<uint32_t *>(blk + o_seed) : nullptr;
    if (rc == SST_OK) {
        const uint8_t *d_raw = blk + o_raw;
        const uint32_t *d_fo = reinterpret_cast<uint32_t *>(blk + o_fo);
        const sst_output *d_out = &d;
        rc = launch_events(ctx, 1, &d_raw, &d_fo, thr, &d_out, st, nullptr, &raw_bytes);
    }
    // counts first, then exactly-sized copies of the cluster arrays
    CU(cudaMemcpyAsync(out->dev_status, d.dev_status, SST_ST_WORDS * 4, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(out->n_clusters, d.n_clusters, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (rc == SST_OK) {
        const size_t k = *out->n_clusters;
        const size_t na = out->dev_status[SST_ST_FLAGS] & (SST_FLAG_CLUSTER_CAP | SST_FLAG_ADC_CAP)
                              ? out->cap_adc
                              : out->dev_status[SST_ST_N_ADC];
        if (k) {
            CU(cudaMemcpyAsync(out->cl_module, d.cl_module, 4 * k, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out->cl_first, d.cl_first, 2 * k, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out->cl_width, d.cl_width, 2 * k, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out->cl_charge, d.cl_charge, 4 * k, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out->cl_bary, d.cl_bary, 4 * k, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out->cl_adc_off, d.cl_adc_off, 4 * k, cudaMemcpyDeviceToHost, st));
            if (out->cl_snr) CU(cudaMemcpyAsync(out->cl_snr, d.cl_snr, 4 * k, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out->cl_adc, d.cl_adc, na, cudaMemcpyDeviceToHost, st));
        }
        if (out->strip_adc) CU(cudaMemcpyAsync(out->strip_adc, d.strip_adc, n, cudaMemcpyDeviceToHost, st));
        if (out->chan_off) CU(cudaMemcpyAsync(out->chan_off, d.chan_off, 4 * nch, cudaMemcpyDeviceToHost, st));
        if (out->chan_len) CU(cudaMemcpyAsync(out->chan_len, d.chan_len, 2 * nch, cudaMemcpyDeviceToHost, st));
        if (out->seed_idx) {
            const size_t ns = std::min<size_t>(out->dev_status[SST_ST_N_SEEDS], out->cap_seeds);
            if (ns) CU(cudaMemcpyAsync(out->seed_idx, d.seed_idx, 4 * ns, cudaMemcpyDeviceToHost, st));
        }
    }
    CU(cudaFreeAsync(blk, st));
    CU(cudaStreamSynchronize(st));
    return rc;
}

namespace {
// A list of copies of one chunk, issued together.
struct CopyList {
    std::vector<void *> dst, src;
    std::vector<size_t> bytes;
    void add(void *d, const void *s, size_t n) {
        if (!n) return;
        dst.push_back(d);
        src.push_back(const_cast<void *>(s));
        bytes.push_back(n);
    }
    cudaError_t run(cudaStream_t st) {
        if (dst.empty()) return cudaSuccess;
        cudaError_t e = cudaSuccess;
        for (size_t i = 0; i < dst.size() && e == cudaSuccess; ++i)
            e = cudaMemcpyAsync(dst[i], src[i], bytes[i], cudaMemcpyDefault, st);
        dst.clear();
        src.clear();
        bytes.clear();
        return e;
    }
};
}  // namespace

sst_status sst_unpack_cluster_host_batch(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                         const uint32_t *raw_bytes, const uint32_t *const *fed_offsets,
                                         const sst_thresholds *thr, const sst_output *outs, void *const *streams,
                                         uint32_t n_streams) {
    if (!ctx || !raw || !raw_bytes || !fed_offsets || !thr || !outs || !streams || n_streams == 0 || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    for (uint32_t e = 0; e < n_events; ++e)
        if (!raw[e] || !fed_offsets[e] || !output_ok(&outs[e]) || !no_device_only_outputs(&outs[e]) ||
            raw_bytes[e] > ctx->cfg.max_raw_bytes)
            return SST_ERR_INVALID_ARG;
    if (n_events == 0) return SST_OK;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    const uint32_t nf = ctx->cfg.n_feds;
    const size_t n = static_cast<size_t>(nf) * kFedStrips, nch = static_cast<size_t>(nf) * kChan;
    auto up = [](size_t b) { return (b + 255) & ~static_cast<size_t>(255); };
    // Chunks of up to kHostChunk events: chunk c runs on streams[c % n_streams] -- upload, one
    // FED-major launch, counts back -- so the uploads, kernels and downloads of neighbouring chunks
    // overlap.  The cluster arrays are then fetched chunk by chunk with exactly-sized
    // copies while later chunks are still being processed.
    auto mapped = [](const void *h, void *&d) {
        cudaPointerAttributes a{};
        if (!h || cudaPointerGetAttributes(&a, h) != cudaSuccess) {
            cudaGetLastError();
            return false;
        }
        d = a.devicePointer;
        return a.type == cudaMemoryTypeHost && a.devicePointer != nullptr;
    };
    struct EvDev { sst_output d; uint8_t *raw; uint32_t *fo; bool direct; };
    struct Chunk { uint32_t e0, n; cudaStream_t st; uint8_t *blk; };
    std::vector<EvDev> dev(n_events);
    std::vector<Chunk> chunks;
    CopyList copies;
    sst_status rc = SST_OK;
    auto CU = [&](cudaError_t e) { if (rc == SST_OK && !cu_ok(ctx, e)) rc = SST_ERR_CUDA; };
    for (uint32_t e0 = 0; e0 < n_events && rc == SST_OK; e0 += kHostChunk) {
        Chunk ck{e0, std::min(kHostChunk, n_events - e0), static_cast<cudaStream_t>(streams[chunks.size() % n_streams]), nullptr};
        // one pooled block per chunk, carved up
        std::vector<size_t> off(ck.n + 1, 0);
        for (uint32_t i = 0; i < ck.n; ++i) {
            const sst_output &o = outs[e0 + i];
            size_t b = up(ctx->cfg.max_raw_bytes) + up((nf + 1) * 4) + up(SST_ST_WORDS * 4) + 256 +
                       up(4ull * o.cap_clusters) * 4 + up(2ull * o.cap_clusters) * 2 + up(o.cap_adc) +
                       (o.cl_snr ? up(4ull * o.cap_clusters) : 0) + (o.strip_adc ? up(n) : 0) +
                       (o.chan_off ? up(4 * nch) : 0) + (o.chan_len ? up(2 * nch) : 0) +
                       (o.seed_idx ? up(4ull * o.cap_seeds) : 0);
            off[i + 1] = off[i] + b;
        }
        CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&ck.blk), off[ck.n], ctx->pool, ck.st));
        if (rc != SST_OK) break;
        const uint8_t *r[kHostChunk];
        const uint32_t *fo[kHostChunk];
        const sst_output *po[kHostChunk];
        for (uint32_t i = 0; i < ck.n; ++i) {
            const sst_output &o = outs[e0 + i];
            EvDev &v = dev[e0 + i];
            uint8_t *q = ck.blk + off[i];
            auto take = [&](size_t bytes) { uint8_t *r0 = q; q += up(bytes); return r0; };
            v.raw = take(ctx->cfg.max_raw_bytes);
            v.fo = reinterpret_cast<uint32_t *>(take((nf + 1) * 4));
            v.d = o;
            // Pinned (mapped) host arrays are written by the emit kernel directly over PCIe: no
            // device copy of the cluster arrays, no count round trip, no per-array download.
            void *m[10] = {};
            v.direct = mapped(o.dev_status, m[0]) && mapped(o.n_clusters, m[1]) && mapped(o.cl_module, m[2]) &&
                       mapped(o.cl_charge, m[3]) && mapped(o.cl_bary, m[4]) && mapped(o.cl_adc_off, m[5]) &&
                       mapped(o.cl_first, m[6]) && mapped(o.cl_width, m[7]) && mapped(o.cl_adc, m[8]) &&
                       (!o.cl_snr || mapped(o.cl_snr, m[9]));
            if (v.direct) {
                v.d.dev_status = static_cast<uint32_t *>(m[0]);
                v.d.n_clusters = static_cast<uint32_t *>(m[1]);
                v.d.cl_module = static_cast<uint32_t *>(m[2]);
                v.d.cl_charge = static_cast<int32_t *>(m[3]);
                v.d.cl_bary = static_cast<float *>(m[4]);
                v.d.cl_adc_off = static_cast<uint32_t *>(m[5]);
                v.d.cl_first = static_cast<uint16_t *>(m[6]);
                v.d.cl_width = static_cast<uint16_t *>(m[7]);
                v.d.cl_adc = static_cast<uint8_t *>(m[8]);
                v.d.cl_snr = o.cl_snr ? static_cast<float *>(m[9]) : nullptr;
            } else {
                v.d.dev_status = reinterpret_cast<uint32_t *>(take(SST_ST_WORDS * 4));
                v.d.n_clusters = reinterpret_cast<uint32_t *>(take(256));
                v.d.cl_module = reinterpret_cast<uint32_t *>(take(4ull * o.cap_clusters));
                v.d.cl_charge = reinterpret_cast<int32_t *>(take(4ull * o.cap_clusters));
                v.d.cl_bary = reinterpret_cast<float *>(take(4ull * o.cap_clusters));
                v.d.cl_adc_off = reinterpret_cast<uint32_t *>(take(4ull * o.cap_clusters));
                v.d.cl_first = reinterpret_cast<uint16_t *>(take(2ull * o.cap_clusters));
                v.d.cl_width = reinterpret_cast<uint16_t *>(take(2ull * o.cap_clusters));
                v.d.cl_adc = take(o.cap_adc);
                v.d.cl_snr = o.cl_snr ? reinterpret_cast<float *>(take(4ull * o.cap_clusters)) : nullptr;
            }
            v.d.strip_adc = o.strip_adc ? take(n) : nullptr;
            v.d.chan_off = o.chan_off ? reinterpret_cast<uint32_t *>(take(4 * nch)) : nullptr;
            v.d.chan_len = o.chan_len ? reinterpret_cast<uint16_t *>(take(2 * nch)) : nullptr;
            v.d.seed_idx = o.seed_idx ? reinterpret_cast<uint32_t *>(take(4ull * o.cap_seeds)) : nullptr;
            copies.add(v.raw, raw[e0 + i], raw_bytes[e0 + i]);
            copies.add(v.fo, fed_offsets[e0 + i], (nf + 1) * 4);
            r[i] = v.raw;
            fo[i] = v.fo;
            po[i] = &v.d;
        }
        CU(copies.run(ck.st));
        if (rc == SST_OK) rc = launch_events(ctx, ck.n, r, fo, thr, po, ck.st, nullptr, raw_bytes + e0);
        for (uint32_t i = 0; i < ck.n; ++i) {
            const sst_output &o = outs[e0 + i];
            if (dev[e0 + i].direct) continue;
            copies.add(o.dev_status, dev[e0 + i].d.dev_status, SST_ST_WORDS * 4);
            copies.add(o.n_clusters, dev[e0 + i].d.n_clusters, 4);
        }
        CU(copies.run(ck.st));
        chunks.push_back(ck);
    }
    // counts are on the host once a chunk's stream has drained: exactly-sized copies of the rest
    for (const Chunk &ck : chunks) {
        CU(cudaStreamSynchronize(ck.st));
        if (rc != SST_OK) break;
        for (uint32_t i = 0; i < ck.n; ++i) {
            const sst_output &o = outs[ck.e0 + i];
            const sst_output &d = dev[ck.e0 + i].d;
            const size_t k = *o.n_clusters;
            const size_t na = o.dev_status[SST_ST_FLAGS] & (SST_FLAG_CLUSTER_CAP | SST_FLAG_ADC_CAP) ? o.cap_adc
                                                                                                     : o.dev_status[SST_ST_N_ADC];
            if (k && !dev[ck.e0 + i].direct) {
                copies.add(o.cl_module, d.cl_module, 4 * k);
                copies.add(o.cl_first, d.cl_first, 2 * k);
                copies.add(o.cl_width, d.cl_width, 2 * k);
                copies.add(o.cl_charge, d.cl_charge, 4 * k);
                copies.add(o.cl_bary, d.cl_bary, 4 * k);
                copies.add(o.cl_adc_off, d.cl_adc_off, 4 * k);
                if (o.cl_snr) copies.add(o.cl_snr, d.cl_snr, 4 * k);
                copies.add(o.cl_adc, d.cl_adc, na);
            }
            if (o.strip_adc) copies.add(o.strip_adc, d.strip_adc, n);
            if (o.chan_off) copies.add(o.chan_off, d.chan_off, 4 * nch);
            if (o.chan_len) copies.add(o.chan_len, d.chan_len, 2 * nch);
            if (o.seed_idx) copies.add(o.seed_idx, d.seed_idx, 4 * std::min<size_t>(o.dev_status[SST_ST_N_SEEDS], o.cap_seeds));
        }
        CU(copies.run(ck.st));
        CU(cudaFreeAsync(ck.blk, ck.st));
    }
    for (const Chunk &ck : chunks) cu_ok(ctx, cudaStreamSynchronize(ck.st));
    return rc;
}

sst_status sst_unpack_cluster_host_packed(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                          const uint32_t *raw_bytes, const uint32_t *const *fed_offsets,
                                          const sst_thresholds *thr, uint32_t cap_clusters, uint32_t cap_adc,
                                          sst_packed_result *results, void *const *streams, uint32_t n_streams) {
    if (!ctx || !raw || !raw_bytes || !fed_offsets || !thr || !results || !streams || n_streams == 0 || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    const size_t block_need = 64 + 20ull * cap_clusters + cap_adc;
    for (uint32_t e = 0; e < n_events; ++e)
        if (!raw[e] || !fed_offsets[e] || !results[e].block || results[e].block_bytes < block_need ||
            raw_bytes[e] > ctx->cfg.max_raw_bytes)
            return SST_ERR_INVALID_ARG;
    if (n_events == 0) return SST_OK;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    const uint32_t nf = ctx->cfg.n_feds;
    auto up = [](size_t b) { return (b + 255) & ~static_cast<size_t>(255); };
    struct Chunk { uint32_t e0, n; cudaStream_t st; uint8_t *blk; };
    std::vector<Chunk> chunks;
    std::vector<uint8_t *> d_block(n_events);
    const size_t per_event = up(ctx->cfg.max_raw_bytes) + up((nf + 1) * 4) + up(block_need);
    sst_status rc = SST_OK;
    auto CU = [&](cudaError_t e) { if (rc == SST_OK && !cu_ok(ctx, e)) rc = SST_ERR_CUDA; };
    sst_output proto{};
    proto.cap_clusters = cap_clusters;
    proto.cap_adc = cap_adc;
    // One download per event, enqueued right behind the launch without waiting for the counts: its
    // size is a guess from the context's running ratio of packed bytes to raw bytes; whatever a
    // guess missed is fetched in a second copy once the counts are on the host.
    float ratio = ctx->packed_ratio.load();
    if (!(ratio > 0.0f)) ratio = 2.2f;
    std::vector<size_t> guess(n_events);
    for (uint32_t e0 = 0; e0 < n_events && rc == SST_OK; e0 += kHostChunk) {
        Chunk ck{e0, std::min(kHostChunk, n_events - e0), static_cast<cudaStream_t>(streams[chunks.size() % n_streams]), nullptr};
        CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&ck.blk), per_event * ck.n, ctx->pool, ck.st));
        if (rc != SST_OK) break;
        const uint8_t *r[kHostChunk];
        const uint32_t *fo[kHostChunk];
        const sst_output *po[kHostChunk];
        uint8_t *pk[kHostChunk];
        for (uint32_t i = 0; i < ck.n; ++i) {
            uint8_t *q = ck.blk + per_event * i;
            uint8_t *d_raw = q;
            uint32_t *d_fo = reinterpret_cast<uint32_t *>(q + up(ctx->cfg.max_raw_bytes));
            d_block[e0 + i] = q + up(ctx->cfg.max_raw_bytes) + up((nf + 1) * 4);
            if (raw_bytes[e0 + i]) CU(cudaMemcpyAsync(d_raw, raw[e0 + i], raw_bytes[e0 + i], cudaMemcpyHostToDevice, ck.st));
            CU(cudaMemcpyAsync(d_fo, fed_offsets[e0 + i], (nf + 1) * 4, cudaMemcpyHostToDevice, ck.st));
            r[i] = d_raw;
            fo[i] = d_fo;
            po[i] = &proto;
            pk[i] = d_block[e0 + i];
        }
        if (rc == SST_OK) rc = launch_events(ctx, ck.n, r, fo, thr, po, ck.st, pk, raw_bytes + e0);
        for (uint32_t i = 0; i < ck.n; ++i) {
            const size_t g = std::min(block_need, 64 + static_cast<size_t>(1.03f * ratio * raw_bytes[e0 + i]) + 4096);
            guess[e0 + i] = g;
            CU(cudaMemcpyAsync(results[e0 + i].block, d_block[e0 + i], g, cudaMemcpyDeviceToHost, ck.st));
        }
        chunks.push_back(ck);
    }
    double sum_need = 0.0, sum_raw = 0.0;
    for (const Chunk &ck : chunks) {
        CU(cudaStreamSynchronize(ck.st));
        if (rc != SST_OK) break;
        for (uint32_t i = 0; i < ck.n; ++i) {
            sst_packed_result &R = results[ck.e0 + i];
            uint8_t *b = static_cast<uint8_t *>(R.block);
            const uint32_t *stw = reinterpret_cast<const uint32_t *>(b);
            const size_t K = std::min(stw[SST_ST_N_CLUSTERS], cap_clusters);
            const size_t na = std::min(stw[SST_ST_N_ADC], cap_adc);
            const size_t need = 64 + 20 * K + na, g = guess[ck.e0 + i];
            if (need > g) CU(cudaMemcpyAsync(b + g, d_block[ck.e0 + i] + g, need - g, cudaMemcpyDeviceToHost, ck.st));
            sum_need += static_cast<double>(need);
            sum_raw += static_cast<double>(raw_bytes[ck.e0 + i]);
            sst_output &v = R.view;
            v = proto;
            v.dev_status = reinterpret_cast<uint32_t *>(b);
            v.n_clusters = reinterpret_cast<uint32_t *>(b + 32);
            v.cl_module = reinterpret_cast<uint32_t *>(b + 64);
            v.cl_charge = reinterpret_cast<int32_t *>(b + 64 + 4 * K);
            v.cl_bary = reinterpret_cast<float *>(b + 64 + 8 * K);
            v.cl_adc_off = reinterpret_cast<uint32_t *>(b + 64 + 12 * K);
            v.cl_first = reinterpret_cast<uint16_t *>(b + 64 + 16 * K);
            v.cl_width = reinterpret_cast<uint16_t *>(b + 64 + 18 * K);
            v.cl_adc = b + 64 + 20 * K;
        }
        CU(cudaFreeAsync(ck.blk, ck.st));
    }
    for (const Chunk &ck : chunks) cu_ok(ctx, cudaStreamSynchronize(ck.st));
    if (rc == SST_OK && sum_raw > 0.0) ctx->packed_ratio.store(static_cast<float>(sum_need / sum_raw));
    return rc;
}

sst_status sst_event_alloc(sst_ctx *ctx, uint64_t bytes, void *stream, void **out_ptr) {
    if (!ctx || !out_ptr || bytes == 0) return SST_ERR_INVALID_ARG;
    *out_ptr = nullptr;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    SST_CU(cudaMallocFromPoolAsync(out_ptr, bytes, ctx->pool, static_cast<cudaStream_t>(stream)));
    return SST_OK;
}

sst_status sst_event_free(sst_ctx *ctx, void *ptr, void *stream) {
    if (!ctx || !ptr) return SST_ERR_INVALID_ARG;
    SST_CU(cudaFreeAsync(ptr, static_cast<cudaStream_t>(stream)));
    return SST_OK;
}

sst_status sst_event_upload(sst_ctx *ctx, const uint8_t *raw, uint32_t raw_bytes,
                            const uint32_t *fed_offsets, void *stream, uint8_t **d_raw,
                            uint32_t **d_fed_offsets) {
    if (!ctx || !raw || !fed_offsets || !d_raw || !d_fed_offsets || raw_bytes > ctx->cfg.max_raw_bytes)
        return SST_ERR_INVALID_ARG;
    *d_raw = nullptr;
    *d_fed_offsets = nullptr;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t fo_bytes = (static_cast<size_t>(ctx->cfg.n_feds) + 1) * sizeof(uint32_t);
    SST_CU(cudaSetDevice(ctx->cfg.device));
    SST_CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(d_raw), ctx->cfg.max_raw_bytes, ctx->pool, st));
    SST_CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(d_fed_offsets), fo_bytes, ctx->pool, st));
    if (raw_bytes) SST_CU(cudaMemcpyAsync(*d_raw, raw, raw_bytes, cudaMemcpyHostToDevice, st));
    SST_CU(cudaMemcpyAsync(*d_fed_offsets, fed_offsets, fo_bytes, cudaMemcpyHostToDevice, st));
    return SST_OK;
}

sst_status sst_event_download(sst_ctx *ctx, void *dst, const void *src, uint64_t bytes, void *stream) {
    if (!ctx || !dst || !src) return SST_ERR_INVALID_ARG;
    if (bytes == 0) return SST_OK;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    SST_CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, static_cast<cudaStream_t>(stream)));
    return SST_OK;
}

sst_status sst_destroy(sst_ctx *ctx) {
    if (!ctx) return SST_ERR_INVALID_ARG;
    cudaSetDevice(ctx->cfg.device);
    cudaDeviceSynchronize();
    for (auto &sl : ctx->slots)
        if (sl.mem) cudaFreeAsync(sl.mem, nullptr);
    for (auto &se : ctx->stream_events) cudaEventDestroy(se.ev);
    cudaDeviceSynchronize();
    if (ctx->calib) cudaFree(ctx->calib);
    if (ctx->calib_orig) cudaFree(ctx->calib_orig);
    if (ctx->bad) cudaFree(ctx->bad);
    if (ctx->geom) cudaFree(ctx->geom);
    if (ctx->chan_info) cudaFree(ctx->chan_info);
    if (ctx->pool) cudaMemPoolDestroy(ctx->pool);
    delete ctx;
    return SST_OK;
}

sst_status sst_trace_read(sst_ctx *ctx, void *stream, uint64_t *out) {
    if (!ctx || !out || !ctx->cfg.trace) return SST_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    SST_CU(cudaSetDevice(ctx->cfg.device));
    std::lock_guard<std::mutex> lock(ctx->slot_mu);
    for (auto &s : ctx->slots) {
        if (s.stream != st || !s.mem) continue;
        uint8_t *tr = s.mem + 256;
        SST_CU(cudaMemcpyAsync(out, tr, SST_TRACE_WORDS * 8, cudaMemcpyDeviceToHost, st));
        SST_CU(cudaMemsetAsync(tr, 0, SST_TRACE_WORDS * 8, st));
        SST_CU(cudaMemsetAsync(tr + 8 * kTrStart, 0xff, 16, st));
        SST_CU(cudaStreamSynchronize(st));
        return SST_OK;
    }
    return SST_ERR_INVALID_ARG;  // nothing was launched on this stream
}

int32_t sst_last_cuda_error(const sst_ctx *ctx) { return ctx ? ctx->last_err.load() : 0; }

const char *sst_status_string(sst_status s) {
    switch (s) {
        case SST_OK: return "SST_OK";
        case SST_ERR_INVALID_ARG: return "SST_ERR_INVALID_ARG";
        case SST_ERR_CUDA: return "SST_ERR_CUDA";
        case SST_ERR_NO_CALIB: return "SST_ERR_NO_CALIB";
        case SST_ERR_BAD_CALIB: return "SST_ERR_BAD_CALIB";
        case SST_ERR_TOO_LARGE: return "SST_ERR_TOO_LARGE";
    }
    return "SST_ERR_UNKNOWN";
}

sst_status sst_get_info(const sst_ctx *ctx, sst_info *info) {
    if (!ctx || !info) return SST_ERR_INVALID_ARG;
    info->smem_bytes = ctx->smem_bytes;
    info->threads = 32 * static_cast<uint32_t>(ctx->wpc);
    info->ctas_per_sm = static_cast<uint32_t>(ctx->ctas_per_sm);
    info->sm_count = static_cast<uint32_t>(ctx->sm_count);
    info->kernels_per_event = ctx->cfg.move_mode == 0 ? 1 : 2;  // (launches with plain outputs)
    info->slot_bytes = ctx->slot_bytes;
    info->events_per_launch = kMaxEv;
    info->pieces = static_cast<uint32_t>(ctx->pieces);
    return SST_OK;
}

}  // extern "C"
