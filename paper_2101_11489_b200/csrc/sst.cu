// sst.cu -- libsst: unpack + three-threshold clustering of strip-tracker FED data on B200.
//
// One persistent kernel per launch, ONE WARP PER FED (a FED is 96 channels x 256
// strips; modules never cross a FED, reading s10).  A CTA is a single warp with a
// ~10 KB shared-memory slot, so ~20 FEDs are in flight per SM and the serial parts of the
// method (the channel-length chain, the run headers) of one FED hide behind the parallel parts
// of the others; there is no block-wide barrier anywhere.  Warps draw FEDs from a ticket
// counter, in (event, FED) order, so a launch takes up to kMaxEv events.
//
// Per FED, everything after the unpack runs in the COMPACT index space of the FED's present
// strips (the structure of arrays of PAPER.md:31 has one entry per recorded strip):
//
//   a1 channel-location map : TMA bulk copy of the FED payload into the slot, the 96-step length
//                             chain walked in shared memory (PAPER.md:31 builds it on the CPU)
//   a2 unpack               : lane per channel: pass 1 validates the run headers and counts, a
//                             warp scan gives every channel its slot range, pass 2 writes the
//                             {strip, adc} lists in ascending strip order
//   a3 flags                : lane per present strip: one 8-byte gather of {noise, gain} (64-byte
//                             L2 fetch), exact >= tests, masks by __ballot_sync, dense SoA scatter
//   a4 seed-index array     : seed mask + ordered compaction; materialised on request
//   a5 expansion/ownership  : bit-parallel flood fill of the seed mask down the link mask, lane
//                             per 32 entries: marks the head of every run that holds a seed, so
//                             each candidate is evaluated once, by (the lane of) its leftmost seed
//   a6 gain corr + accept   : q = min(254, floor(adc/gain + .5)) in float32; lane per candidate:
//                             Q^2 >= t^2 * sum n^2 with the double sum taken left to right
//   a7 ordered output       : FED aggregate published in one 64-bit word, every FED sums the
//                             words of its predecessors (one round trip), lane per cluster emit
//
// FEDs whose payload or lists exceed the slot run the same code on a pooled global scratch.
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
#include <vector>

#include "sst.h"

namespace {

constexpr int kChan = 96;
constexpr int kStrip = 256;
constexpr int kFedStrips = kChan * kStrip;  // 24576
constexpr int kMaxEv = 8;                   // events per launch
constexpr int kQCap = 256;                  // candidate / cluster queue (entries)
constexpr int kWide = 48;                   // candidates wider than this are summed by the warp
constexpr int kU = 4;                       // mask words per batch of the flag pass (loads in flight)
constexpr uint32_t kFull = 0xffffffffu;
constexpr uint32_t kMaxFeds = 4096;

// Published FED aggregate, one 64-bit word: epoch (12 bits, never 0) << 52 | overrun << 51 |
// malformed channels (7) << 44 | seeds (15) << 29 | cluster ADC bytes (15) << 14 | clusters (14).
// A word counts only if its epoch is the launch's; the host clears the array when the epoch wraps.
constexpr int kShEpoch = 52, kShOver = 51, kShMalf = 44, kShSeed = 29, kShAdc = 14;
constexpr uint32_t kEpochMax = 4095;

struct EventDesc {
    const uint8_t *raw;
    const uint32_t *fed_offsets;
    sst_output out;
};

struct KParams {
    const float2 *calib;     // {noise (+inf at bad strips), gain} per strip
    const uint2 *chan_info;  // {module id, first channel | end channel << 8 of the module}
    unsigned long long *fed_state;  // [kMaxEv][n_feds]
    unsigned long long *ticket;     // monotone counter; this launch owns [ticket_base, +total+grid)
    unsigned long long ticket_base;
    // global scratch of the slow path, one slice set per event
    float *g_noise;
    uint16_t *g_strip;
    uint8_t *g_adc;
    uint32_t *g_mask;  // 4 arrays of g_mwords per event
    uint32_t g_ents, g_mwords;
    double tcl2;
    float t_ch, t_seed;
    uint32_t max_raw_bytes, n_feds, n_events, epoch, slot_bytes;
    unsigned long long *phase_clk;  // debug builds only (SST_PHASE_TIMING)
    EventDesc ev[kMaxEv];
};

// per-warp shared memory: fixed header, then the slot (payload stage, later the lists and masks)
struct __align__(16) Hdr {
    unsigned long long mbar;
    uint32_t chan_off[kChan];  // FED-local byte offset of the channel's first run byte
    uint16_t chan_len[kChan];
    uint16_t queue[kQCap];
};
constexpr uint32_t kHdrBytes = (sizeof(Hdr) + 127u) & ~127u;

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
__device__ __forceinline__ unsigned long long ld_state(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_state(unsigned long long *p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// L2 residency.  The calibration (8 B per strip, 86.5 MB for 440 FEDs) is read by every event and
// fits the L2 set-aside that sst_create reserves, while raw data and outputs stream through once:
// calibration loads carry an evict_last policy, everything else that touches HBM evict_first.
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
// Calibration gather.  On B200 a plain load that misses L2 pulls the whole 128-byte line from
// DRAM; the .L2::64B qualifier halves that (measured, profiles/r01_v4.md), and nothing is reused
// through L1.
__device__ __forceinline__ float2 ld_calib(const float2 *p, unsigned long long pol) {
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.L2::64B.v2.f32 {%0,%1}, [%2], %3;"
                 : "=f"(v.x), "=f"(v.y)
                 : "l"(p), "l"(pol));
    return v;
}
// streaming stores of the outputs
__device__ __forceinline__ void st_stream(uint4 *p, uint4 v, unsigned long long pol) {
    asm volatile("st.global.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w), "l"(pol)
                 : "memory");
}
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
    return (a > p) || (a == p && e <= 0.0f);
}
// min(254, floor(fl32(fl32(adc / gain) + 0.5)))  (IEEE RN division and add, no contraction)
__device__ __forceinline__ uint32_t gain_correct(float adc, float gain) {
    const float u = __fadd_rn(__fdiv_rn(adc, gain), 0.5f);
    const float fl = floorf(u);
    return fl >= 254.0f ? 254u : static_cast<uint32_t>(fl);
}

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ unsigned long long warp_sum64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_d(double v) {
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

// Entry i is "linked" when it continues the cluster candidate of entry i-1 (both active, strips
// adjacent inside one module).  The last entry of the run that contains entry i: one before the
// next unlinked entry.  link[] has zero sentinel words after the last used word.
__device__ __forceinline__ int run_end(const uint32_t *link, int i) {
    int w = i >> 5;
    const int b = i & 31;
    uint32_t nl = ~link[w] & (b == 31 ? 0u : (kFull << (b + 1)));
    while (nl == 0) nl = ~link[++w];
    return (w << 5) + __ffs(nl) - 2;
}

// x |= every entry from which a set entry of x is reached by walking up through linked entries
// (bit j of l: entry j continues entry j-1).  Kogge-Stone fill, five doubling steps.
__device__ __forceinline__ uint32_t fill_down(uint32_t x, uint32_t l) {
    x |= (x & l) >> 1;
    l &= l << 1;
    x |= (x & l) >> 2;
    l &= l << 2;
    x |= (x & l) >> 4;
    l &= l << 4;
    x |= (x & l) >> 8;
    l &= l << 8;
    x |= (x & l) >> 16;
    return x;
}

// Cluster acceptance for a narrow candidate, one lane: Q^2 >= t_cl^2 * n2 with n2 the double sum
// of noise^2 taken strictly left to right (reading s15; noise^2 is exact in double, so
// the fused multiply-add below rounds exactly like the oracle's separate multiply and add).
__device__ __forceinline__ bool accept_serial(const uint8_t *q, const float *noise, int l, int w, double tcl2) {
    int Q = 0;
    double n2 = 0.0;
#pragma unroll 1
    for (int i = 0; i < w; ++i) {
        Q += q[l + i];
        const double d = static_cast<double>(noise[l + i]);
        n2 = __fma_rn(d, d, n2);
    }
    const double lhs = static_cast<double>(Q) * static_cast<double>(Q);
    return lhs >= __dmul_rn(tcl2, n2);
}

// The same decision for a wide candidate by the whole warp.  A pairwise double sum differs from
// the sequential one by at most ~w*2^-52 relative; the decision is taken from it only when the
// two sides are further apart than that, otherwise lane 0 redoes the sum sequentially.
__device__ __noinline__ bool accept_warp(const uint8_t *q, const float *noise, int l, int w, double tcl2, int lane) {
    uint32_t Q = 0;
    double n2p = 0.0;
#pragma unroll 1
    for (int i = lane; i < w; i += 32) {
        Q += q[l + i];
        const double d = static_cast<double>(noise[l + i]);
        n2p += d * d;
    }
    Q = warp_sum(Q);
    n2p = warp_sum_d(n2p);
    const double lhs = static_cast<double>(Q) * static_cast<double>(Q);
    const double rhs = tcl2 * n2p;
    int ok = lhs >= rhs;
    if (!(fabs(lhs - rhs) > rhs * static_cast<double>(w) * 0x1p-50)) {
        if (lane == 0) {
            double n2 = 0.0;
#pragma unroll 1
            for (int i = 0; i < w; ++i) {
                const double d = static_cast<double>(noise[l + i]);
                n2 = __fma_rn(d, d, n2);
            }
            ok = lhs >= __dmul_rn(tcl2, n2);
        }
        ok = __shfl_sync(kFull, ok, 0);
    }
    return ok != 0;
}

// optional output: cluster S/N = Q / sqrt(sum noise^2), sequential double sum
__device__ __noinline__ float cluster_snr(const float *noise, int l, int w, int Q) {
    double n2 = 0.0;
#pragma unroll 1
    for (int i = 0; i < w; ++i) {
        const double d = static_cast<double>(noise[l + i]);
        n2 = __fma_rn(d, d, n2);
    }
    return static_cast<float>(static_cast<double>(Q) / sqrt(n2));
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
__device__ __forceinline__ void walk_chain_speculative(const uint8_t *stage, uint32_t clamp, uint32_t *chan_off,
                                                       uint16_t *chan_len) {
    uint32_t pos = 0;
#pragma unroll 8
    for (int c = 0; c < kChan; ++c) {
        const uint32_t a = min(pos, clamp);
        const uint32_t l16 = stage[a] | (static_cast<uint32_t>(stage[a + 1]) << 8);
        chan_off[c] = pos + 2;
        chan_len[c] = static_cast<uint16_t>(l16);
        pos += 2 + l16;
    }
}

// a2 pass 1: validate one channel's run list (reading s2b) and count its strips.
// Returns false for a malformed channel.
__device__ __forceinline__ bool scan_runs(const uint8_t *rp, uint32_t off, uint32_t len_bytes, uint32_t &n_strips) {
    uint32_t q = off, next_free = 0, within = 0;
    const uint32_t qend = off + len_bytes;
    bool ok = true;
#pragma unroll 1
    while (q < qend) {
        if (q + 2 > qend) { ok = false; break; }
        const uint32_t first = rp[q];
        uint32_t len = rp[q + 1];
        if (len == 0) len = 256;  // reading s2
        if (first < next_free || first + len > kStrip || q + 2 + len > qend) { ok = false; break; }
        next_free = first + len;
        q += 2 + len;
        within += len;
    }
    n_strips = within;
    return ok;
}

#ifdef SST_PHASE_TIMING
#define SST_MARK(k) do { if (lane == 0 && p.phase_clk) p.phase_clk[static_cast<size_t>(ticket) * 16 + (k)] = clock64(); } while (0)
#else
#define SST_MARK(k) do { } while (0)
#endif

struct FedCtx {
    uint32_t ticket, ev, f;
    uint32_t fo0;                 // the FED's start offset as given (reported in chan_off)
    uint32_t fed_start, fed_size;  // what is read: [fed_start, +fed_size), empty for a bad FED
    uint32_t overrun, n_malformed;
    uint32_t P;
    uint32_t off[3], len[3], base[3];  // of channels lane, lane+32, lane+64
    uint32_t opens;                    // bit k: channel lane+32k opens a module
};

// ------------------------------------------------------------------------------ lists -> clusters
// Everything after pass 1, on the FED's lists of present strips, by one warp.  kFast: lists and
// masks live in the warp's shared-memory slot (LDS/STS) and the payload is staged there; else
// lists and masks live in this FED's slice of the global scratch and rp is a generic pointer.
template <bool kFast>
__device__ __forceinline__ void fed_lists(const KParams &p, Hdr &h, uint8_t *slot, const uint8_t *rp,
                                          const FedCtx &c, const int lane, uint32_t &next_ticket) {
    const uint32_t f = c.f, P = c.P, ticket = c.ticket;
    const EventDesc &E = p.ev[c.ev];
    const sst_output &o = E.out;
    const uint32_t nw = (P + 31) >> 5;  // mask words in use
    const uint32_t lt = (1u << lane) - 1u;
    (void)ticket;

    float *noise_l;
    uint16_t *strip_l;
    uint8_t *adc_l;
    uint32_t *mS, *mL, *mH, *mX;
    if (kFast) {
        const uint32_t A = (max((c.fed_size + 15u) & ~15u, 4u * P) + 15u) & ~15u;
        noise_l = reinterpret_cast<float *>(slot);  // overlays the payload once the lists are built
        strip_l = reinterpret_cast<uint16_t *>(slot + A);
        adc_l = slot + A + 2u * P;
        mS = reinterpret_cast<uint32_t *>(slot + ((A + 3u * P + 3u) & ~3u));
        mL = mS + (nw + 2);
        mH = mL + (nw + 2);
        mX = mH + (nw + 2);
    } else {
        const size_t eb = static_cast<size_t>(c.ev) * p.g_ents;
        const uint32_t slice = ((c.fed_start + 15u) & ~15u) + 16u * f;
        noise_l = p.g_noise + eb + slice;
        strip_l = p.g_strip + eb + slice;
        adc_l = p.g_adc + eb + slice;
        mS = p.g_mask + static_cast<size_t>(c.ev) * 4u * p.g_mwords + (slice >> 5) + 4u * f;
        mL = mS + p.g_mwords;
        mH = mL + p.g_mwords;
        mX = mH + p.g_mwords;
    }
    uint8_t *const dense = o.strip_adc ? o.strip_adc + static_cast<size_t>(f) * kFedStrips : nullptr;

    // ---------------------------------------------------------------- a2 pass 2: lane per channel
    // writes {strip, adc} in ascending strip order; bit 15 of a strip id marks strip 0 of a channel
    // that opens a module (nothing links across it)
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        uint32_t q = c.off[k], e = c.base[k];
        const uint32_t qend = q + c.len[k];
        const uint32_t g0 = static_cast<uint32_t>(lane + 32 * k) * kStrip;
        const uint32_t open_bit = ((c.opens >> k) & 1u) << 15;
#pragma unroll 1
        while (q < qend) {
            const uint32_t first = rp[q];
            uint32_t len = rp[q + 1];
            if (len == 0) len = 256;
            // most runs hold one or two strips; on the fast path the second byte is read
            // unconditionally (it is inside the slot or its 16-byte tail pad)
            const uint32_t b0 = rp[q + 2], b1 = (kFast || len > 1) ? rp[q + 3] : 0u;
            const uint32_t sid = g0 + first;
            strip_l[e] = static_cast<uint16_t>(first == 0 ? sid | open_bit : sid);
            adc_l[e] = static_cast<uint8_t>(b0);
            if (len > 1) {
                strip_l[e + 1] = static_cast<uint16_t>(sid + 1u);
                adc_l[e + 1] = static_cast<uint8_t>(b1);
            }
#pragma unroll 1
            for (uint32_t i = 2; i < len; ++i) {
                strip_l[e + i] = static_cast<uint16_t>(sid + i);
                adc_l[e + i] = rp[q + 2 + i];
            }
            e += len;
            q += 2 + len;
        }
        __syncwarp();
    }
    __syncwarp();  // lists complete; the payload is dead from here on

    SST_MARK(4);
    // ---------------------------------------------------------------- a3: active / seed flags
    // lane per entry, a warp covers one mask word per step, so the masks come from ballots; kU
    // words per batch keep kU calibration gathers in flight per lane
    const float2 *cal = p.calib + static_cast<size_t>(f) * kFedStrips;
    const unsigned long long pol_last = policy_evict_last(), pol_first = policy_evict_first();
    {
        uint32_t carry_sv = 0xffffu, carry_act = 0;
        uint32_t filled = 0;  // the dense output is zero up to here (multiple of 16)
        const bool dense16 = (reinterpret_cast<uintptr_t>(dense) & 15u) == 0;
        auto fill_to = [&](uint32_t upto) {
            if (dense16) {
#pragma unroll 1
                for (uint32_t b = filled + 16u * lane; b < upto; b += 512u)
                    st_stream(reinterpret_cast<uint4 *>(dense + b), make_uint4(0, 0, 0, 0), pol_first);
            } else {
#pragma unroll 1
                for (uint32_t b = filled + lane; b < upto; b += 32u) dense[b] = 0;
            }
            filled = upto;
            __syncwarp();
        };
#pragma unroll 1
        for (uint32_t w0 = 0; w0 < nw; w0 += kU) {
            uint32_t sv[kU], av[kU];
            float2 cv[kU];
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                const uint32_t i = (w0 + j) * 32u + lane;
                const bool valid = i < P;
                sv[j] = valid ? strip_l[i] : 0xffffu;
                av[j] = valid ? adc_l[i] : 0u;
            }
#pragma unroll
            for (int j = 0; j < kU; ++j)
                cv[j] = av[j] ? ld_calib(cal + (sv[j] & 0x7fffu), pol_last) : make_float2(INFINITY, 1.0f);
            if (dense) {
                // zero-fill the dense output up to the last strip of this batch (to the FED's end in
                // the last batch), just ahead of the scatter below: both hit the same L2 lines
                const uint32_t i_last = min(P, (w0 + kU) * 32u) - 1u;
                fill_to((w0 + kU) * 32u >= P ? static_cast<uint32_t>(kFedStrips)
                                             : ((strip_l[i_last] & 0x7fffu) + 16u) & ~15u);
            }
#pragma unroll
            for (int j = 0; j < kU; ++j) {
                if (w0 + j >= nw) break;  // warp-uniform
                const uint32_t i = (w0 + j) * 32u + lane;
                const bool valid = sv[j] != 0xffffu;
                const uint32_t s15 = sv[j] & 0x7fffu;
                if (dense && valid) st_stream(dense + s15, av[j], pol_first);
                const float af = static_cast<float>(av[j]);
                const bool is_act = av[j] != 0 && ge_exact(af, p.t_ch, cv[j].x);
                const bool is_seed = is_act && ge_exact(af, p.t_seed, cv[j].x);
                uint32_t p_sv = __shfl_up_sync(kFull, sv[j], 1);
                uint32_t p_act = __shfl_up_sync(kFull, static_cast<uint32_t>(is_act), 1);
                if (lane == 0) { p_sv = carry_sv; p_act = carry_act; }
                // this entry continues the candidate of the previous one
                const bool is_link = is_act && p_act && !(sv[j] & 0x8000u) && s15 == (p_sv & 0x7fffu) + 1u;
                const uint32_t wa = __ballot_sync(kFull, is_act);
                const uint32_t ws = __ballot_sync(kFull, is_seed);
                const uint32_t wl = __ballot_sync(kFull, is_link);
                if (valid) {
                    noise_l[i] = cv[j].x;
                    if (is_act) adc_l[i] = static_cast<uint8_t>(gain_correct(af, cv[j].y));
                }
                if (lane == 0) {
                    mS[w0 + j] = ws;
                    mL[w0 + j] = wl;
                    mH[w0 + j] = wa & ~wl;  // heads: active entries that start a candidate
                }
                carry_sv = __shfl_sync(kFull, sv[j], 31);
                carry_act = __shfl_sync(kFull, static_cast<uint32_t>(is_act), 31);
            }
        }
        if (dense && filled < static_cast<uint32_t>(kFedStrips)) fill_to(kFedStrips);  // a FED without strips
        if (lane < 2) {  // zero sentinels behind the last word
            mS[nw + lane] = 0;
            mL[nw + lane] = 0;
            mH[nw + lane] = 0;
            mX[nw + lane] = 0;
        }
    }
    __syncwarp();

    SST_MARK(5);
    // ---------------------------------------------------------------- a4/a5: seeds -> candidates
    // lane per mask word: X = entries with a seed at or above them in their run (flood fill of
    // the seed mask down the links); a head in X starts a candidate that holds a seed.  Runs that
    // cross a word boundary hand the fill to the word below until nothing changes.
    uint32_t n_seed = 0;
#pragma unroll 1
    for (uint32_t w = lane; w < nw; w += 32) {
        const uint32_t s = mS[w];
        n_seed += __popc(s);
        mX[w] = fill_down(s, mL[w]);
    }
    __syncwarp();
    for (;;) {
        bool changed = false;
#pragma unroll 1
        for (uint32_t w = lane; w < nw; w += 32) {
            const uint32_t cin = mX[w + 1] & mL[w + 1] & 1u;
            const uint32_t x = mX[w];
            if (cin && !(x >> 31)) {
                mX[w] = fill_down(x | 0x80000000u, mL[w]);
                changed = true;
            }
        }
        __syncwarp();
        if (!__any_sync(kFull, changed)) break;
    }
#pragma unroll 1
    for (uint32_t w = lane; w < nw; w += 32) mH[w] &= mX[w];
    __syncwarp();

    SST_MARK(6);
    // ---------------------------------------------------------------- a6: lane per candidate
    // candidates are queued in order, kQCap at a time; a rejected one clears its head bit, so mH
    // ends as the mask of accepted clusters
    uint32_t my_cl = 0, my_adc = 0;
    {
        uint32_t qn = 0;
        auto flush = [&]() {
            __syncwarp();
#pragma unroll 1
            for (uint32_t c0 = 0; c0 < qn; c0 += 32) {
                const uint32_t ci = c0 + lane;
                const bool have = ci < qn;
                int hd = 0, wd = 0;
                bool ok = false;
                if (have) {
                    hd = h.queue[ci];
                    wd = run_end(mL, hd) - hd + 1;
                    if (wd <= kWide) ok = accept_serial(adc_l, noise_l, hd, wd, p.tcl2);
                }
                uint32_t widem = __ballot_sync(kFull, have && wd > kWide);
                while (widem) {
                    const int src = __ffs(widem) - 1;
                    widem &= widem - 1;
                    const int hh = __shfl_sync(kFull, hd, src), ww = __shfl_sync(kFull, wd, src);
                    const bool r = accept_warp(adc_l, noise_l, hh, ww, p.tcl2, lane);
                    if (lane == src) ok = r;
                }
                if (have) {
                    if (ok) {
                        ++my_cl;
                        my_adc += wd;
                    } else {
                        atomicAnd(&mH[hd >> 5], ~(1u << (hd & 31)));
                    }
                }
                __syncwarp();
            }
            qn = 0;
        };
#pragma unroll 1
        for (uint32_t w = 0; w < nw; ++w) {
            const uint32_t hs = mH[w];
            const uint32_t n = __popc(hs);
            if (!n) continue;
            if (qn + n > static_cast<uint32_t>(kQCap)) flush();
            if ((hs >> lane) & 1u) h.queue[qn + __popc(hs & lt)] = static_cast<uint16_t>(w * 32u + lane);
            qn += n;
        }
        flush();
    }
    const uint32_t fed_cl = warp_sum(my_cl), fed_adc = warp_sum(my_adc), fed_seed = warp_sum(n_seed);

    SST_MARK(7);
    // ---------------------------------------------------------------- a7: publish, sum predecessors
    unsigned long long *const st = p.fed_state + static_cast<size_t>(c.ev) * p.n_feds;
    if (lane == 0) {
        st_state(st + f, (static_cast<unsigned long long>(p.epoch) << kShEpoch) |
                             (static_cast<unsigned long long>(c.overrun) << kShOver) |
                             (static_cast<unsigned long long>(c.n_malformed) << kShMalf) |
                             (static_cast<unsigned long long>(fed_seed) << kShSeed) |
                             (static_cast<unsigned long long>(fed_adc) << kShAdc) | fed_cl);
        // next FED of this warp: the ticket arrives while the look-back and the emit run
        next_ticket = static_cast<uint32_t>(atomicAdd(p.ticket, 1ull) - p.ticket_base);
    }
    // clusters | ADC bytes << 32 ; seeds | malformed << 32 (20 bits) | overrun << 52 (n_feds <= 4096)
    unsigned long long accA = 0, accB = 0;
#pragma unroll 1
    for (uint32_t j0 = 0; j0 < f; j0 += 128) {  // warp-uniform control flow: the lanes poll together
        unsigned long long v[4];
        bool need[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const uint32_t j = j0 + 32u * u + lane;
            need[u] = j < f;
            v[u] = need[u] ? ld_state(st + j) : 0ull;
        }
        for (;;) {
            bool ok = true;
#pragma unroll
            for (int u = 0; u < 4; ++u) ok = ok && (!need[u] || (v[u] >> kShEpoch) == p.epoch);
            if (__all_sync(kFull, ok)) break;
            __nanosleep(100);  // some predecessor has not published in this launch yet
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (need[u] && (v[u] >> kShEpoch) != p.epoch) v[u] = ld_state(st + j0 + 32u * u + lane);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (need[u]) {
                accA += (v[u] & 0x3fffull) | (((v[u] >> kShAdc) & 0x7fffull) << 32);
                accB += ((v[u] >> kShSeed) & 0x7fffull) | (((v[u] >> kShMalf) & 0x7full) << 32) |
                        (((v[u] >> kShOver) & 1ull) << 52);
            }
    }
    accA = warp_sum64(accA);
    accB = warp_sum64(accB);
    const uint32_t b_cl = static_cast<uint32_t>(accA), b_adc = static_cast<uint32_t>(accA >> 32);
    const uint32_t b_seed = static_cast<uint32_t>(accB), b_malf = static_cast<uint32_t>(accB >> 32) & 0xfffffu,
                   b_over = static_cast<uint32_t>(accB >> 52);

    SST_MARK(8);
    // ---------------------------------------------------------------- a4: seed-index array (on request)
    if (o.seed_idx) {
        uint32_t k0 = b_seed;
#pragma unroll 1
        for (uint32_t w = 0; w < nw; ++w) {
            const uint32_t sw = mS[w];
            if ((sw >> lane) & 1u) {
                const uint32_t k = k0 + __popc(sw & lt);
                if (k < o.cap_seeds) o.seed_idx[k] = f * kFedStrips + (strip_l[w * 32u + lane] & 0x7fffu);
            }
            k0 += __popc(sw);
        }
    }
    // ---------------------------------------------------------------- a7: emit, (module, first strip) order
    {
        uint32_t qn = 0, run_cl = b_cl, run_adc = b_adc;
        const uint2 *cinfo = p.chan_info + static_cast<size_t>(f) * kChan;
        auto flush = [&]() {
            __syncwarp();
#pragma unroll 1
            for (uint32_t c0 = 0; c0 < qn; c0 += 32) {
                const uint32_t ci = c0 + lane;
                const bool have = ci < qn;
                int hd = 0, wd = 0;
                if (have) {
                    hd = h.queue[ci];
                    wd = run_end(mL, hd) - hd + 1;
                }
                const uint32_t incl = warp_incl_scan(static_cast<uint32_t>(wd), lane);
                const uint32_t k_cl = run_cl + ci, k_adc = run_adc + incl - wd;
                run_adc += __shfl_sync(kFull, incl, 31);
                if (have && k_cl < o.cap_clusters && k_adc + wd <= o.cap_adc) {
                    int Q = 0;
                    long long M = 0;
#pragma unroll 1
                    for (int j = 0; j < wd; ++j) {
                        const int q = adc_l[hd + j];
                        Q += q;
                        M += static_cast<long long>(j) * q;
                        st_stream(o.cl_adc + k_adc + j, static_cast<uint32_t>(q), pol_first);
                    }
                    const uint32_t st0 = strip_l[hd] & 0x7fffu;
                    const uint2 cm = __ldg(cinfo + (st0 >> 8));
                    const int first = static_cast<int>(st0) - static_cast<int>(cm.y & 0xffu) * kStrip;
                    st_stream(o.cl_module + k_cl, cm.x, pol_first);
                    st_stream(o.cl_first + k_cl, static_cast<uint32_t>(first), pol_first);
                    st_stream(o.cl_width + k_cl, static_cast<uint32_t>(wd), pol_first);
                    st_stream(o.cl_charge + k_cl, Q, pol_first);
                    // barycenter in float32: first + M/Q is good to ~2e-7 relative (tolerance 1e-6)
                    st_stream(o.cl_bary + k_cl,
                              __fadd_rn(static_cast<float>(first), __fdiv_rn(static_cast<float>(M), static_cast<float>(Q))),
                              pol_first);
                    st_stream(o.cl_adc_off + k_cl, k_adc, pol_first);
                    if (o.cl_snr) o.cl_snr[k_cl] = cluster_snr(noise_l, hd, wd, Q);
                } else if (have) {
                    // the first cluster that does not fit reports how many were written
                    const bool prev_fits = k_cl == 0 || (k_cl - 1 < o.cap_clusters && k_adc <= o.cap_adc);
                    if (prev_fits) *o.n_clusters = k_cl;
                }
                __syncwarp();
            }
            run_cl += qn;
            qn = 0;
        };
#pragma unroll 1
        for (uint32_t w = 0; w < nw; ++w) {
            const uint32_t hs = mH[w];
            const uint32_t n = __popc(hs);
            if (!n) continue;
            if (qn + n > static_cast<uint32_t>(kQCap)) flush();
            if ((hs >> lane) & 1u) h.queue[qn + __popc(hs & lt)] = static_cast<uint16_t>(w * 32u + lane);
            qn += n;
        }
        flush();
    }
    if (f == p.n_feds - 1 && lane == 0) {  // event totals = prefix of the last FED + its own
        const uint32_t n_cl = b_cl + fed_cl, n_adc = b_adc + fed_adc, n_mal = b_malf + c.n_malformed,
                       n_over = b_over + c.overrun;
        uint32_t flags = 0;
        if (n_cl > o.cap_clusters) flags |= SST_FLAG_CLUSTER_CAP;
        if (n_adc > o.cap_adc) flags |= SST_FLAG_ADC_CAP;
        if (n_mal) flags |= SST_FLAG_MALFORMED;
        if (n_over) flags |= SST_FLAG_OVERRUN;
        if (!(flags & (SST_FLAG_CLUSTER_CAP | SST_FLAG_ADC_CAP))) *o.n_clusters = n_cl;
        o.dev_status[SST_ST_FLAGS] = flags;
        o.dev_status[SST_ST_N_MALFORMED] = n_mal;
        o.dev_status[SST_ST_N_CLUSTERS] = n_cl;
        o.dev_status[SST_ST_N_ADC] = n_adc;
        o.dev_status[SST_ST_N_OVERRUN] = n_over;
        o.dev_status[SST_ST_N_SEEDS] = b_seed + fed_seed;
        o.dev_status[6] = 0;
        o.dev_status[7] = 0;
    }
    SST_MARK(9);
}

// bytes of slot a FED needs on the fast path: payload stage (later noise), lists, four masks
__device__ __forceinline__ uint32_t slot_need(uint32_t fed_size, uint32_t P) {
    const uint32_t A = (max((fed_size + 15u) & ~15u, 4u * P) + 15u) & ~15u;
    return ((A + 3u * P + 3u) & ~3u) + 16u * (((P + 31u) >> 5) + 2u);
}

// ------------------------------------------------------------------------------ one FED, one warp
__device__ __forceinline__ void process_fed(const KParams &p, Hdr &h, uint8_t *slot, const uint32_t ticket,
                                            const int lane, uint32_t &mbar_phase, uint32_t &next_ticket) {
    FedCtx c;
    c.ticket = ticket;
    c.ev = ticket / p.n_feds;
    c.f = ticket - c.ev * p.n_feds;
    const uint32_t f = c.f;
    const EventDesc &E = p.ev[c.ev];
    const sst_output &o = E.out;

    SST_MARK(0);
    // ---------------------------------------------------------------- a1: stage the FED payload
    // lanes 0/1 fetch the two offsets; lane 0 starts the bulk copy
    const uint32_t fo = lane < 2 ? E.fed_offsets[f + lane] : 0u;
    const uint32_t fo0 = __shfl_sync(kFull, fo, 0), fo1 = __shfl_sync(kFull, fo, 1);
    const bool valid = fo0 <= fo1 && fo1 <= p.max_raw_bytes;
    c.fo0 = fo0;
    c.fed_start = valid ? fo0 : 0u;
    c.fed_size = valid ? fo1 - fo0 : 0u;
    c.overrun = valid ? 0u : 1u;
    const bool staged = c.fed_size <= p.slot_bytes && ((c.fed_start | c.fed_size) & 15u) == 0 &&
                        (reinterpret_cast<uintptr_t>(E.raw) & 15u) == 0;
    __syncwarp();  // every lane is done with the slot of the previous FED
    if (staged && c.fed_size && lane == 0) {
        fence_proxy_async();  // earlier generic-proxy accesses to the slot before the async write
        mbar_expect_tx(&h.mbar, c.fed_size);
        bulk_g2s(slot, E.raw + c.fed_start, c.fed_size, &h.mbar, policy_evict_first());
    }
    // meanwhile: fetch the module map
    c.opens = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t ch = lane + 32 * k;
        const uint2 ci = __ldg(p.chan_info + static_cast<size_t>(f) * kChan + ch);
        if ((ci.y & 0xffu) == ch) c.opens |= 1u << k;
    }
    const uint8_t *rp = staged ? slot : E.raw + c.fed_start;
    if (staged && c.fed_size) {
        mbar_wait(&h.mbar, mbar_phase);  // every lane waits: async-proxy writes visible to all readers
        mbar_phase ^= 1u;
    }

    SST_MARK(1);
    // ---------------------------------------------------------------- a1: walk the length chain
    if (staged) {
        if (lane == 0) walk_chain_speculative(slot, p.slot_bytes - 2u, h.chan_off, h.chan_len);
        __syncwarp();
        // validate the speculative chain: channels from the first bad one on are empty
        uint32_t bad = 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            c.off[k] = h.chan_off[lane + 32 * k];
            c.len[k] = h.chan_len[lane + 32 * k];
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
        if (lane == 0) over = walk_chain_checked(rp, c.fed_size, c.overrun != 0, h.chan_off, h.chan_len) ? 1u : 0u;
        c.overrun = __shfl_sync(kFull, over, 0);
        __syncwarp();
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            c.off[k] = h.chan_off[lane + 32 * k];
            c.len[k] = h.chan_len[lane + 32 * k];
        }
    }

    SST_MARK(2);
    // ---------------------------------------------------------------- a2 pass 1: run headers
    // lane per channel: validate the run list, count the strips
    uint32_t cnt[3];
    c.n_malformed = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t ch = lane + 32 * k;
        if (o.chan_off) o.chan_off[f * kChan + ch] = c.fo0 + c.off[k];
        if (o.chan_len) o.chan_len[f * kChan + ch] = static_cast<uint16_t>(c.len[k]);
        uint32_t n_strips = 0;
        const bool ok = staged ? scan_runs(slot, c.off[k], c.len[k], n_strips) : scan_runs(rp, c.off[k], c.len[k], n_strips);
        __syncwarp();
        cnt[k] = ok ? n_strips : 0u;
        if (!ok) c.len[k] = 0;  // a malformed channel contributes no strips
        c.n_malformed += __popc(__ballot_sync(kFull, !ok));
    }
    // exclusive scan of the 96 counts
    uint32_t run = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const uint32_t inc = warp_incl_scan(cnt[k], lane);
        c.base[k] = run + inc - cnt[k];
        run += __shfl_sync(kFull, inc, 31);
    }
    c.P = run;  // present strips of the FED

    SST_MARK(3);
    if (staged && slot_need(c.fed_size, c.P) <= p.slot_bytes)
        fed_lists<true>(p, h, slot, slot, c, lane, next_ticket);
    else
        fed_lists<false>(p, h, slot, rp, c, lane, next_ticket);
}

// ------------------------------------------------------------------------------ the kernel
// A CTA is one warp.  Warps draw (event, FED) tickets until the launch's work is used up.
__global__ void __launch_bounds__(32, 24) sst_event_kernel(const __grid_constant__ KParams p) {
    extern __shared__ __align__(128) uint8_t smem_raw[];
    Hdr &h = *reinterpret_cast<Hdr *>(smem_raw);
    uint8_t *slot = smem_raw + kHdrBytes;
    const int lane = threadIdx.x;
    if (lane == 0) {
        mbar_init(&h.mbar, 1);
        fence_proxy_async();
    }
    __syncwarp();
    const uint32_t total = p.n_events * p.n_feds;
    uint32_t mbar_phase = 0;
    uint32_t ticket = 0;
    if (lane == 0) ticket = static_cast<uint32_t>(atomicAdd(p.ticket, 1ull) - p.ticket_base);
    ticket = __shfl_sync(kFull, ticket, 0);
    while (ticket < total) {
        uint32_t next_ticket = 0;
        process_fed(p, h, slot, ticket, lane, mbar_phase, next_ticket);
        ticket = __shfl_sync(kFull, next_ticket, 0);
    }
}

}  // namespace

// ====================================================================================== host
struct sst_ctx {
    sst_config cfg{};
    cudaMemPool_t pool = nullptr;
    float2 *calib = nullptr;
    uint2 *chan_info = nullptr;
    bool has_calib = false;
    std::atomic<int32_t> last_err{0};
    int sm_count = 0;
    int ctas_per_sm = 0;
    uint32_t slot_bytes = 0;  // shared-memory slot of one warp (one FED)
    uint32_t smem_bytes = 0;  // header + slot
    // per-stream scratch (ticket counter, FED states, slow-path lists), taken from the pool on a
    // stream's first launch and kept: stream order makes reuse safe, the epoch and the running
    // ticket base make clearing unnecessary
    struct Slot { cudaStream_t stream; uint8_t *mem; uint32_t epoch; unsigned long long ticket_base; };
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

bool thresholds_ok(const sst_thresholds *t) {
    const float v[3] = {t->channel, t->seed, t->cluster};
    for (float x : v)
        if (!std::isfinite(x) || !(x > 0.0f)) return false;
    return true;
}

bool output_ok(const sst_output *o) {
    return o && o->n_clusters && o->dev_status && o->cl_module && o->cl_first && o->cl_width &&
           o->cl_charge && o->cl_bary && o->cl_adc_off && o->cl_adc && !(o->seed_idx == nullptr && o->cap_seeds != 0);
}

#ifdef SST_PHASE_TIMING
unsigned long long *g_phase_clk = nullptr;
#endif

struct ScratchLayout {
    size_t ents, mwords, state_bytes, o_ticket, o_state, o_noise, o_mask, o_strip, o_adc, total;
};
ScratchLayout scratch_layout(const sst_ctx *ctx) {
    ScratchLayout L{};
    const uint32_t nf = ctx->cfg.n_feds;
    auto up = [](size_t b) { return (b + 255) & ~static_cast<size_t>(255); };
    L.ents = (static_cast<size_t>(ctx->cfg.max_raw_bytes) + 16ull * nf + 64 + 31) & ~static_cast<size_t>(31);
    L.mwords = L.ents / 32 + 4ull * nf + 16;
    L.state_bytes = sizeof(unsigned long long) * nf * kMaxEv;
    L.o_ticket = 0;
    L.o_state = 256;
    L.o_noise = L.o_state + up(L.state_bytes);
    L.o_mask = L.o_noise + up(4 * L.ents * kMaxEv);
    L.o_strip = L.o_mask + up(4 * 4 * L.mwords * kMaxEv);
    L.o_adc = L.o_strip + up(2 * L.ents * kMaxEv);
    L.total = L.o_adc + up(L.ents * kMaxEv);
    return L;
}

// Launches one kernel for `n` (<= kMaxEv) events on `st`.
sst_status launch_events(sst_ctx *ctx, uint32_t n, const uint8_t *const *raw, const uint32_t *const *fed_offsets,
                         const sst_thresholds *thr, const sst_output *const *outs, cudaStream_t st) {
    const uint32_t nf = ctx->cfg.n_feds;
    const ScratchLayout L = scratch_layout(ctx);
    const uint32_t total = n * nf;
    const uint32_t capacity = static_cast<uint32_t>(ctx->sm_count * ctx->ctas_per_sm);
    const uint32_t grid = std::min(total, capacity);
    uint8_t *blk = nullptr;
    uint32_t epoch = 0;
    unsigned long long ticket_base = 0;
    {
        std::lock_guard<std::mutex> lock(ctx->slot_mu);
        sst_ctx::Slot *sl = nullptr;
        for (auto &s : ctx->slots)
            if (s.stream == st) sl = &s;
        if (!sl) {
            SST_CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&blk), L.total, ctx->pool, st));
            SST_CU(cudaMemsetAsync(blk, 0, L.o_noise, st));  // ticket counter and states
            ctx->slots.push_back({st, blk, 0u, 0ull});
            sl = &ctx->slots.back();
        }
        if (sl->epoch == kEpochMax) {  // epoch wraps: stale words of 4095 launches ago must not match
            SST_CU(cudaMemsetAsync(sl->mem + L.o_state, 0, L.state_bytes, st));
            sl->epoch = 0;
        }
        sl->epoch += 1;
        blk = sl->mem;
        epoch = sl->epoch;
        ticket_base = sl->ticket_base;
        sl->ticket_base += static_cast<unsigned long long>(total) + grid;  // every warp draws one ticket too many
    }
    KParams kp{};
    kp.calib = ctx->calib;
    kp.chan_info = ctx->chan_info;
    kp.ticket = reinterpret_cast<unsigned long long *>(blk + L.o_ticket);
    kp.ticket_base = ticket_base;
    kp.fed_state = reinterpret_cast<unsigned long long *>(blk + L.o_state);
    kp.g_noise = reinterpret_cast<float *>(blk + L.o_noise);
    kp.g_mask = reinterpret_cast<uint32_t *>(blk + L.o_mask);
    kp.g_strip = reinterpret_cast<uint16_t *>(blk + L.o_strip);
    kp.g_adc = blk + L.o_adc;
    kp.g_ents = static_cast<uint32_t>(L.ents);
    kp.g_mwords = static_cast<uint32_t>(L.mwords);
    kp.tcl2 = static_cast<double>(thr->cluster) * static_cast<double>(thr->cluster);  // exact
    kp.t_ch = thr->channel;
    kp.t_seed = thr->seed;
    kp.max_raw_bytes = ctx->cfg.max_raw_bytes;
    kp.n_feds = nf;
    kp.n_events = n;
    kp.epoch = epoch;
    kp.slot_bytes = ctx->slot_bytes;
#ifdef SST_PHASE_TIMING
    kp.phase_clk = g_phase_clk;
#endif
    for (uint32_t e = 0; e < n; ++e) {
        kp.ev[e].raw = raw[e];
        kp.ev[e].fed_offsets = fed_offsets[e];
        kp.ev[e].out = *outs[e];
    }
    sst_event_kernel<<<grid, 32, ctx->smem_bytes, st>>>(kp);
    SST_CU(cudaGetLastError());
    return SST_OK;
}

}  // namespace

extern "C" {

#ifdef SST_PHASE_TIMING
void sst_debug_set_phase_clk(unsigned long long *p) { g_phase_clk = p; }
#endif

sst_status sst_create(const sst_config *cfg, sst_ctx **out_ctx) {
    if (out_ctx) *out_ctx = nullptr;
    if (!cfg || !out_ctx || cfg->n_feds == 0 || cfg->n_feds > kMaxFeds || cfg->max_raw_bytes == 0)
        return SST_ERR_INVALID_ARG;
    sst_ctx *ctx = new (std::nothrow) sst_ctx();
    if (!ctx) return SST_ERR_INVALID_ARG;
    ctx->cfg = *cfg;
    if (ctx->cfg.max_events_in_flight == 0) ctx->cfg.max_events_in_flight = 8;
    auto fail = [&](sst_status s) {
        if (ctx->calib) cudaFree(ctx->calib);
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
    if (cudaMalloc(&ctx->chan_info, static_cast<size_t>(cfg->n_feds) * kChan * sizeof(uint2)) !=
        cudaSuccess)
        return fail(SST_ERR_CUDA);
    // shared-memory slot of one warp: sized for the largest FED the configuration expects (FEDs
    // that do not fit take the slow path through the global scratch)
    {
        const double m = static_cast<double>(cfg->max_raw_bytes) / cfg->n_feds;  // mean payload bound
        const uint32_t p_hint = cfg->fed_strips_hint ? std::min(cfg->fed_strips_hint, static_cast<uint32_t>(kFedStrips))
                                                     : static_cast<uint32_t>(0.55 * m) + 32u;
        const uint32_t r_hint = (static_cast<uint32_t>(std::min(1.15 * m + 64.0, 65536.0)) + 15u) & ~15u;
        const uint32_t A = (std::max(r_hint, 4u * p_hint) + 15u) & ~15u;
        uint32_t need = ((A + 3u * p_hint + 3u) & ~3u) + 16u * (((p_hint + 31u) >> 5) + 2u);
        need = (need + 127u) & ~127u;
        ctx->slot_bytes = std::min(std::max(need, 2048u), 200u * 1024u);
        ctx->smem_bytes = kHdrBytes + ctx->slot_bytes + 16u;  // tail pad, see pass 2
    }
    if (cudaFuncSetAttribute(sst_event_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(ctx->smem_bytes)) != cudaSuccess)
        return fail(SST_ERR_CUDA);
    cudaFuncSetAttribute(sst_event_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    {
        // L2 set-aside for the calibration (read by every event with an evict_last policy): the
        // device maximum (79 of 126 MB on B200).  A device-wide limit; failure is not fatal.
        int max_persist = 0;
        if (cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, cfg->device) == cudaSuccess &&
            max_persist > 0)
            cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, static_cast<size_t>(max_persist));
        cudaGetLastError();
    }
    cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, cfg->device);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->ctas_per_sm, sst_event_kernel, 32,
                                                      ctx->smem_bytes) != cudaSuccess || ctx->ctas_per_sm < 1)
        return fail(SST_ERR_CUDA);
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
    for (size_t g = 0; g < n; ++g) {
        if (bad[g]) {
            // a bad strip is never active: noise = +inf fails every >= test; gain is never used
            packed[g] = make_float2(INFINITY, 1.0f);
        } else {
            if (!std::isfinite(gain[g]) || !(gain[g] > 0.0f) || !std::isfinite(noise[g]) || !(noise[g] > 0.0f))
                return SST_ERR_BAD_CALIB;
            packed[g] = make_float2(noise[g], gain[g]);
        }
    }
    SST_CU(cudaSetDevice(ctx->cfg.device));
    SST_CU(cudaMemcpy(ctx->calib, packed.data(), n * sizeof(float2), cudaMemcpyHostToDevice));
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

sst_status sst_unpack_cluster(sst_ctx *ctx, const uint8_t *raw, const uint32_t *fed_offsets,
                              const sst_thresholds *thr, const sst_output *out, void *stream) {
    if (!ctx || !raw || !fed_offsets || !thr || !output_ok(out) || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    return launch_events(ctx, 1, &raw, &fed_offsets, thr, &out, static_cast<cudaStream_t>(stream));
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
    // the events of one stream go into launches of up to kMaxEv events each
    for (uint32_t s = 0; s < n_streams && s < n_events; ++s) {
        const uint8_t *r[kMaxEv];
        const uint32_t *fo[kMaxEv];
        const sst_output *o[kMaxEv];
        uint32_t n = 0;
        for (uint32_t e = s; e < n_events; e += n_streams) {
            r[n] = raw[e];
            fo[n] = fed_offsets[e];
            o[n] = &outs[e];
            if (++n == kMaxEv || e + n_streams >= n_events) {
                const sst_status rc = launch_events(ctx, n, r, fo, thr, o, static_cast<cudaStream_t>(streams[s]));
                if (rc != SST_OK) return rc;
                n = 0;
            }
        }
    }
    return SST_OK;
}

sst_status sst_unpack_cluster_host(sst_ctx *ctx, const uint8_t *raw, uint32_t raw_bytes,
                                   const uint32_t *fed_offsets, const sst_thresholds *thr,
                                   const sst_output *out, void *stream) {
    if (!ctx || !raw || !fed_offsets || !thr || !output_ok(out) || !thresholds_ok(thr))
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
        rc = launch_events(ctx, 1, &d_raw, &d_fo, thr, &d_out, st);
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

sst_status sst_destroy(sst_ctx *ctx) {
    if (!ctx) return SST_ERR_INVALID_ARG;
    cudaSetDevice(ctx->cfg.device);
    cudaDeviceSynchronize();
    for (auto &sl : ctx->slots) cudaFreeAsync(sl.mem, nullptr);
    cudaDeviceSynchronize();
    if (ctx->calib) cudaFree(ctx->calib);
    if (ctx->chan_info) cudaFree(ctx->chan_info);
    if (ctx->pool) cudaMemPoolDestroy(ctx->pool);
    delete ctx;
    return SST_OK;
}

int32_t sst_last_cuda_error(const sst_ctx *ctx) { return ctx ? ctx->last_err.load() : 0; }

const char *sst_status_string(sst_status s) {
    switch (s) {
        case SST_OK: return "SST_OK";
        case SST_ERR_INVALID_ARG: return "SST_ERR_INVALID_ARG";
        case SST_ERR_CUDA: return "SST_ERR_CUDA";
        case SST_ERR_NO_CALIB: return "SST_ERR_NO_CALIB";
        case SST_ERR_BAD_CALIB: return "SST_ERR_BAD_CALIB";
    }
    return "SST_ERR_UNKNOWN";
}

sst_status sst_get_info(const sst_ctx *ctx, sst_info *info) {
    if (!ctx || !info) return SST_ERR_INVALID_ARG;
    info->smem_bytes = ctx->smem_bytes;
    info->threads = 32;
    info->ctas_per_sm = static_cast<uint32_t>(ctx->ctas_per_sm);
    info->sm_count = static_cast<uint32_t>(ctx->sm_count);
    info->kernels_per_event = 1;
    info->slot_bytes = ctx->slot_bytes;
    info->events_per_launch = kMaxEv;
    return SST_OK;
}

}  // extern "C"
