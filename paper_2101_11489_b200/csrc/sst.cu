// sst.cu -- libsst: unpack + three-threshold clustering of strip-tracker FED data on B200.
//
// One fused kernel per event, one CTA per FED (a FED is 96 channels x 256 strips;
// modules never cross a FED, reading s10).  After the unpack everything runs in the
// COMPACT index space of the FED's present strips (the structure of arrays of PAPER.md:31 has
// one entry per recorded strip), kept in shared memory:
//
//   a1 channel-location map : TMA bulk copy of the FED payload to smem, 96-step length chain
//                             walked in smem (PAPER.md:31 builds this map on the CPU)
//   a2 unpack               : thread per channel; pass 1 walks the run headers (validate, count),
//                             a 96-wide scan gives every channel its slot range, pass 2 streams
//                             the payload bytes into {strip, adc} lists in ascending strip order
//                             and scatters the ADCs into the zero-filled dense output
//   a3 flags                : lane per present strip: one 8-byte gather of {noise, gain},
//                             exact >= tests, masks built with __ballot_sync (no atomics)
//   a4 seed-index array     : seed mask + block scan; materialised on request
//   a5 expansion/ownership  : lane per seed: bit scans over a "linked to the previous entry"
//                             mask; only the leftmost seed of a run goes on
//   a6 gain corr + accept   : q = min(254, floor(adc/gain + .5)) in float32, Q^2 >= t^2 * sum n^2
//   a7 ordered output       : block scan + look-back over per-FED aggregates, lane per cluster
//
// FEDs whose payload or strip count exceed the smem budgets use the same code on slices of a
// pooled global scratch buffer.  No tensor cores: nothing here is a contraction.
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

constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kChan = 96;
constexpr int kStrip = 256;
constexpr int kFedStrips = kChan * kStrip;  // 24576
constexpr int kListCap = 4096;              // present strips per FED kept in smem
constexpr int kRawCap = 4 * kListCap;       // FED payload staged in smem (region reused for noise)
constexpr int kMaskWords = kListCap / 32 + 1;
constexpr int kRunCap = 2048;               // run-table slots (FED payloads up to ~6 KB)
constexpr int kInline = 8;                  // runs up to this length are copied by one thread
constexpr int kLongQ = 96;
constexpr int kWide = 32;                   // clusters wider than this are summed by a warp
constexpr int kWideQ = 32;
enum { M_ACT = 0, M_SEED, M_BRK, M_LINK, M_ACC, M_WTOT, M_COUNT };

// per-FED aggregate published for the look-back (one 64-bit word)
// look-back state, two 64-bit words per FED, living in a per-stream scratch that is never cleared:
// every word carries the 8-bit epoch of the call that wrote it and counts only if that matches.
// Word 0: status (bits 62-63: 1 = aggregate, 2 = inclusive prefix) | epoch (bits 54-61) | clusters
// (26 bits) | ADC bytes << 26 (28 bits).  Word 1, aggregate only: ready (bit 63) | epoch (bits 55-62)
// | seeds (20 bits) | malformed channels << 20 (7 bits) | overrun << 27.
constexpr unsigned long long kStA = 1ull << 62, kStP = 2ull << 62, kStMask = (1ull << 54) - 1;
constexpr int kShEp0 = 54, kShEp1 = 55, kShAdc = 26;
constexpr int kShMalf = 20, kShOvr = 27;
constexpr unsigned long long kReady = 1ull << 63;
constexpr uint32_t kMaxFeds = 4096;  // keeps event totals inside the 26/28-bit prefix fields

struct __align__(128) Smem {
    union {                       // the payload is dead once the lists are built
        uint8_t raw[kRawCap];     // FED payload (TMA destination)
        float noise[kListCap];    // noise of entry i
    } u;
    uint16_t strip[kListCap];     // FED-local strip id of entry i, ascending
    uint8_t adc[kListCap];        // raw ADC, replaced by the corrected ADC at active entries
    uint32_t mask[M_COUNT][kMaskWords];
    alignas(16) uint32_t runs[kRunCap];  // one record per run, slot = (runs of earlier channels' bound) + ordinal
    uint32_t mod_id[kChan];
    uint32_t chan_off[kChan];     // FED-local byte offset of the first run byte
    uint16_t chan_len[kChan];
    uint16_t chan_base[kChan];    // first list entry of the channel
    uint16_t slot_base[kChan + 1];
    uint8_t mod_lo[kChan], mod_hi[kChan];  // first channel / end channel of the channel's module
    uint32_t okmask[3];
    uint32_t wscan[2][kWarps];
    uint32_t red[5][kWarps];
    uint32_t wide_q[kWideQ];
    uint16_t long_q[kLongQ];
    unsigned long long mbar;
    uint32_t wide_count, long_count;
    uint32_t fed_start, fed_size, in_smem, overrun;
};

struct KParams {
    const uint8_t *raw;
    const uint32_t *fed_offsets;
    const float2 *calib;     // {noise (+inf at bad strips), gain} per strip
    const uint2 *chan_info;  // {module id, first channel | end channel << 8 of the module}
    unsigned long long *fed_state;
    // global scratch for FEDs that do not fit the smem lists (sliced by FED offset)
    uint16_t *g_strip;
    uint8_t *g_adc;
    float *g_noise;
    uint32_t *g_mask;  // M_COUNT arrays of g_mask_words
    uint32_t g_mask_words;
    double tcl2;
    float t_ch, t_seed;
    uint32_t max_raw_bytes, n_feds;
    uint32_t epoch;  // 1..255, changes on every use of the scratch
    sst_output out;
    unsigned long long *phase_clk;  // debug builds only (SST_PHASE_TIMING)
};

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
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_addr(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// TMA bulk copy global -> shared (non-tensor form), completion on an mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes,
                                         unsigned long long *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_addr(dst)),
        "l"(src), "r"(bytes), "r"(smem_addr(bar))
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

// ------------------------------------------------------------------------------ arithmetic
// adc >= t * noise decided in exact arithmetic with float32 only: t*n = p + e exactly (FMA).
// noise = +inf (bad strip) gives p = inf, e = NaN -> false.
__device__ __forceinline__ bool ge_exact(float a, float t, float n) {
    const float p = __fmul_rn(t, n);
    const float e = __fmaf_rn(t, n, -p);
    return (a > p) || (a == p && e <= 0.0f);
}
// min(254, floor(fl32(fl32(adc / gain) + 0.5)))  (IEEE RN division and add, no contraction)
__device__ __noinline__ uint32_t gain_correct(uint32_t adc, float gain) {
    const float u = __fadd_rn(__fdiv_rn(static_cast<float>(adc), gain), 0.5f);
    const float fl = floorf(u);
    return fl >= 254.0f ? 254u : static_cast<uint32_t>(fl);
}

__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Entry i is "linked" when it continues the cluster candidate of entry i-1 (both active, strips
// adjacent inside one module).  The last entry of the run that contains entry i: one before the
// next unlinked entry.  link[] has a zero sentinel word after the last used word.
__device__ __forceinline__ int run_end(const uint32_t *link, int i) {
    int w = i >> 5;
    const int b = i & 31;
    uint32_t nl = ~link[w] & (b == 31 ? 0u : (0xffffffffu << (b + 1)));
    while (nl == 0) nl = ~link[++w];
    return (w << 5) + __ffs(nl) - 2;
}

// Cluster acceptance for a narrow candidate, one thread: Q^2 >= t_cl^2 * n2 with n2 the double
// sum of noise^2 taken strictly left to right (reading s15).
__device__ __forceinline__ bool accept_serial(const uint8_t *q, const float *noise, int l, int w, double tcl2) {
    int Q = 0;
    double n2 = 0.0;
    #pragma unroll 1
    for (int i = 0; i < w; ++i) {
        Q += q[l + i];
        const double d = static_cast<double>(noise[l + i]);
        n2 = __dadd_rn(n2, __dmul_rn(d, d));
    }
    const double lhs = static_cast<double>(Q) * static_cast<double>(Q);
    return lhs >= __dmul_rn(tcl2, n2);
}

// The same decision for a wide candidate by one warp.  A pairwise double sum differs from the
// sequential one by at most ~w*2^-52 relative; the decision is taken from it only when the two
// sides are further apart than that, otherwise lane 0 redoes the sum sequentially.
__device__ __noinline__ bool accept_warp(const uint8_t *q, const float *noise, int l, int w, double tcl2,
                                         int lane) {
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
                n2 = __dadd_rn(n2, __dmul_rn(d, d));
            }
            ok = lhs >= __dmul_rn(tcl2, n2);
        }
        ok = __shfl_sync(0xffffffffu, ok, 0);
    }
    return ok != 0;
}

// optional output: cluster S/N = Q / sqrt(sum noise^2), sequential double sum
__device__ __noinline__ float cluster_snr(const float *noise, int l, int w, int Q) {
    double n2 = 0.0;
#pragma unroll 1
    for (int i = 0; i < w; ++i) {
        const double d = static_cast<double>(noise[l + i]);
        n2 = __dadd_rn(n2, __dmul_rn(d, d));
    }
    return static_cast<float>(static_cast<double>(Q) / sqrt(n2));
}

// ------------------------------------------------------------------------------ raw payload
// Loops that read the raw bytes are instantiated on the smem stage (LDS) and on the generic
// global pointer (oversized or unaligned FEDs).

// a1: the channel-length chain of one FED, checked as it goes (generic path).
__device__ __forceinline__ bool walk_chain_checked(const uint8_t *rp, uint32_t fed_size, bool over, uint32_t *chan_off,
                                                   uint16_t *chan_len, uint16_t *slot_base) {
    uint32_t pos = 0, slots = 0;
    int c = 0;
    if (!over) {
        #pragma unroll 1
        for (; c < kChan; ++c) {
            if (pos + 2 > fed_size) break;
            const uint32_t l16 = rp[pos] | (static_cast<uint32_t>(rp[pos + 1]) << 8);
            if (pos + 2 + l16 > fed_size) break;
            chan_off[c] = pos + 2;
            chan_len[c] = static_cast<uint16_t>(l16);
            slot_base[c] = static_cast<uint16_t>(min(slots, 0xffffu));
            slots += l16 / 3;
            pos += 2 + l16;
        }
    }
    over = c < kChan;
    #pragma unroll 1
    for (; c < kChan; ++c) {  // channels behind an overrun are empty, recorded at the FED end
        chan_off[c] = fed_size;
        chan_len[c] = 0;
        slot_base[c] = static_cast<uint16_t>(min(slots, 0xffffu));
    }
    slot_base[kChan] = static_cast<uint16_t>(min(slots, 0xffffu));
    return over;
}

// a1, smem stage: the same chain walked speculatively -- no bounds checks inside the serial
// loop (addresses wrap inside the stage), the 96 results are validated in parallel afterwards.
__device__ __forceinline__ void walk_chain_speculative(const uint8_t *stage, uint32_t *chan_off, uint16_t *chan_len,
                                                       uint16_t *slot_base) {
    uint32_t pos = 0, slots = 0;
#pragma unroll 4
    for (int c = 0; c < kChan; ++c) {
        const uint32_t a = pos & (kRawCap - 1);
        const uint32_t l16 = stage[a] | (static_cast<uint32_t>(stage[(a + 1) & (kRawCap - 1)]) << 8);
        chan_off[c] = pos + 2;
        chan_len[c] = static_cast<uint16_t>(l16);
        slot_base[c] = static_cast<uint16_t>(min(slots, 0xffffu));
        slots += l16 / 3;
        pos += 2 + l16;
    }
    slot_base[kChan] = static_cast<uint16_t>(min(slots, 0xffffu));
}

// a2 pass 1: validate one channel's run list (reading s2b), count its strips and, when
// the run table is in use, leave one record per run: strips before | first << 8 | (len-1) << 16
// | channel << 24 | valid << 31.  Returns false for a malformed channel.
__device__ __forceinline__ bool scan_runs(const uint8_t *rp, uint32_t off, uint32_t len_bytes, uint32_t chan,
                                          uint32_t *slots, uint32_t &n_runs, uint32_t &n_strips) {
    uint32_t q = off, next_free = 0, k = 0, within = 0;
    const uint32_t qend = off + len_bytes;
    bool ok = true;
    #pragma unroll 1
    while (q < qend) {
        if (q + 2 > qend) { ok = false; break; }
        const uint32_t first = rp[q];
        uint32_t len = rp[q + 1];
        if (len == 0) len = 256;  // reading s2
        if (first < next_free || first + len > kStrip || q + 2 + len > qend) { ok = false; break; }
        if (slots) slots[k] = within | (first << 8) | ((len - 1) << 16) | (chan << 24) | 0x80000000u;
        next_free = first + len;
        q += 2 + len;
        within += len;
        ++k;
    }
    n_runs = k;
    n_strips = within;
    return ok;
}

// a2 pass 2, fallback without the run table: stream one (validated) channel byte by byte.
__device__ __forceinline__ void stream_channel(const uint8_t *rp, uint32_t off, uint32_t len_bytes, uint32_t k,
                                               int chan, uint16_t *strip_l, uint8_t *adc_l, uint8_t *dense) {
    uint32_t rem = 0, tgt = 0, hdr = 0;
    const uint32_t qend = off + len_bytes;
    #pragma unroll 1
    for (uint32_t q = off; q < qend; ++q) {
        const uint32_t b = rp[q];
        if (rem) {
            strip_l[k] = static_cast<uint16_t>(chan * kStrip + tgt);
            adc_l[k] = static_cast<uint8_t>(b);
            if (dense) dense[chan * kStrip + tgt] = static_cast<uint8_t>(b);
            ++k; ++tgt; --rem;
        } else if (!hdr) {
            tgt = b;
            hdr = 1;
        } else {
            rem = b ? b : 256u;
            hdr = 0;
        }
    }
}

#ifdef SST_PHASE_TIMING
#define SST_MARK(k) do { if (threadIdx.x == 0 && p.phase_clk) p.phase_clk[blockIdx.x * 16 + (k)] = clock64(); } while (0)
#else
#define SST_MARK(k) do { } while (0)
#endif

// ------------------------------------------------------------------------------ lists -> clusters
// Everything after the channel walk, on the FED's lists of present strips.  kSmem = true: lists
// and masks in shared memory (LDS/STS); false: in this FED's slice of the global scratch.
template <bool kSmem>
__device__ __noinline__ void lists_to_clusters(const KParams &p, Smem &s, const uint8_t *rp, const uint32_t P,
                                                  const bool table_ok, const uint32_t n_slots,
                                                  const uint32_t n_malformed, const uint32_t my_off,
                                                  const uint32_t my_len, const uint32_t my_base) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t f = blockIdx.x;
    const sst_output &o = p.out;
    const uint32_t nw = (P + 31) >> 5;  // mask words in use
    const uint32_t slice = ((s.fed_start + 15u) & ~15u) + 16u * f;
    uint16_t *const strip_l = kSmem ? s.strip : p.g_strip + slice;
    uint8_t *const adc_l = kSmem ? s.adc : p.g_adc + slice;
    float *const noise_l = kSmem ? s.u.noise : p.g_noise + slice;
    uint32_t *const mbase = kSmem ? &s.mask[0][0] : p.g_mask + (slice >> 5) + 2u * f;
    const uint32_t mstride = kSmem ? static_cast<uint32_t>(kMaskWords) : p.g_mask_words;
#define MASK(k) (mbase + (k) * mstride)
    uint8_t *const dense = o.strip_adc ? o.strip_adc + static_cast<size_t>(f) * kFedStrips : nullptr;

    // ---------------------------------------------------------------- a2 pass 2: thread per run
    if (table_ok) {
        #pragma unroll 1
        for (uint32_t slot = tid; slot < n_slots; slot += kThreads) {
            const uint32_t rec = s.runs[slot];
            if (!(rec >> 31)) continue;
            const uint32_t c = (rec >> 24) & 127u, within = rec & 255u, first = (rec >> 8) & 255u,
                           len = ((rec >> 16) & 255u) + 1u;
            if (len > kInline) {
                const uint32_t qi = atomicAdd(&s.long_count, 1u);
                if (qi < kLongQ) { s.long_q[qi] = static_cast<uint16_t>(slot); continue; }
            }
            const uint32_t src = s.chan_off[c] + within + 2u * (slot - s.slot_base[c] + 1u);
            const uint32_t dst = s.chan_base[c] + within, g = c * kStrip + first;
            #pragma unroll 1
            for (uint32_t i = 0; i < len; ++i) {
                const uint8_t b = rp[src + i];
                strip_l[dst + i] = static_cast<uint16_t>(g + i);
                adc_l[dst + i] = b;
                if (dense) dense[g + i] = b;
            }
        }
        __syncthreads();
        const uint32_t nq = min(s.long_count, static_cast<uint32_t>(kLongQ));
        #pragma unroll 1
        for (uint32_t e = warp; e < nq; e += kWarps) {  // long runs: one warp each, lane per byte
            const uint32_t slot = s.long_q[e], rec = s.runs[slot];
            const uint32_t c = (rec >> 24) & 127u, within = rec & 255u, first = (rec >> 8) & 255u,
                           len = ((rec >> 16) & 255u) + 1u;
            const uint32_t src = s.chan_off[c] + within + 2u * (slot - s.slot_base[c] + 1u);
            const uint32_t dst = s.chan_base[c] + within, g = c * kStrip + first;
            #pragma unroll 1
            for (uint32_t i = lane; i < len; i += 32) {
                const uint8_t b = rp[src + i];
                strip_l[dst + i] = static_cast<uint16_t>(g + i);
                adc_l[dst + i] = b;
                if (dense) dense[g + i] = b;
            }
        }
    } else if (tid < kChan && my_len) {
        stream_channel(rp, my_off, my_len, my_base, tid, strip_l, adc_l, dense);
    }
    __syncthreads();  // lists complete; the payload (smem union) is dead from here on

    SST_MARK(5);
    // ---------------------------------------------------------------- a3: active / seed flags
    // lane per entry; a warp covers one mask word per step, so the masks come from ballots
    const float2 *cal = p.calib + static_cast<size_t>(f) * kFedStrips;
    #pragma unroll 1
    for (uint32_t base = 0; base < nw * 32; base += kThreads * 2) {
        uint32_t idx[2], sv[2], av[2], sp[2];
        float2 cv[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            idx[j] = base + j * kThreads + tid;
            const bool valid = idx[j] < P;
            sv[j] = valid ? strip_l[idx[j]] : 0u;
            av[j] = valid ? adc_l[idx[j]] : 0u;
            sp[j] = (valid && idx[j] > 0) ? strip_l[idx[j] - 1] : 0xffffu;
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) cv[j] = av[j] ? __ldg(cal + sv[j]) : make_float2(INFINITY, 1.0f);
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            if ((base + j * kThreads + warp * 32) >= nw * 32) continue;  // warp-uniform
            const float af = static_cast<float>(av[j]);
            const bool is_act = av[j] != 0 && ge_exact(af, p.t_ch, cv[j].x);
            const bool is_seed = is_act && ge_exact(af, p.t_seed, cv[j].x);
            const uint32_t ch = sv[j] >> 8;
            // a new candidate must start here if the previous entry is not the strip to the left
            // or this strip opens a module
            const bool is_brk = sv[j] != sp[j] + 1u || ((sv[j] & 255u) == 0 && s.mod_lo[ch] == ch);
            if (idx[j] < P) {
                noise_l[idx[j]] = cv[j].x;
                if (is_act) adc_l[idx[j]] = static_cast<uint8_t>(gain_correct(av[j], cv[j].y));
            }
            const uint32_t wa = __ballot_sync(0xffffffffu, is_act);
            const uint32_t ws = __ballot_sync(0xffffffffu, is_seed);
            const uint32_t wb = __ballot_sync(0xffffffffu, is_brk);
            if (lane == 0) {
                const uint32_t w = idx[j] >> 5;
                MASK(M_ACT)[w] = wa; MASK(M_SEED)[w] = ws; MASK(M_BRK)[w] = wb;
            }
        }
    }
    __syncthreads();
    #pragma unroll 1
    for (uint32_t w = tid; w <= nw; w += kThreads) {  // link mask (+ zero sentinel word), clear acc
        uint32_t lk = 0;
        if (w < nw) {
            const uint32_t a = MASK(M_ACT)[w];
            const uint32_t carry = w ? (MASK(M_ACT)[w - 1] >> 31) : 0u;
            lk = a & ((a << 1) | carry) & ~MASK(M_BRK)[w];
        } else {
            MASK(M_SEED)[w] = 0;
        }
        MASK(M_LINK)[w] = lk;
        MASK(M_ACC)[w] = 0;
        MASK(M_WTOT)[w] = 0;
    }
    __syncthreads();

    SST_MARK(6);
    // ---------------------------------------------------------------- a5 + a6: lane per seed
    const uint32_t *const m_link = MASK(M_LINK);
    const uint32_t *const m_seed = MASK(M_SEED);
    uint32_t *const m_acc = MASK(M_ACC);
    #pragma unroll 1
    for (uint32_t i = tid; i < nw * 32; i += kThreads) {
        const int w = i >> 5, b = i & 31;
        const uint32_t sw = m_seed[w];
        if (!((sw >> b) & 1u)) continue;
        // left: the run starts at the nearest unlinked entry at or below i; a seed in between owns it
        int ww = w;
        uint32_t nl = ~m_link[w] & (0xffffffffu >> (31 - b));
        uint32_t sd = sw & ((1u << b) - 1u);
        bool owner = true;
        while (nl == 0) {  // entry 0 is never linked, so this ends
            if (sd) { owner = false; break; }
            --ww;
            nl = ~m_link[ww];
            sd = m_seed[ww];
        }
        if (!owner) continue;
        const int hb = 31 - __clz(nl);
        if (sd >> hb) continue;  // leftmost-seed ownership: another seed emits this cluster
        const int l = (ww << 5) + hb;
        const int wd = run_end(m_link, i) - l + 1;
        if (wd > kWide) {
            const uint32_t slot = atomicAdd(&s.wide_count, 1u);
            if (slot < kWideQ) {
                s.wide_q[slot] = static_cast<uint32_t>(l) | (static_cast<uint32_t>(wd) << 16);
                continue;
            }
        }
        if (accept_serial(adc_l, noise_l, l, wd, p.tcl2)) {
            atomicOr(&m_acc[l >> 5], 1u << (l & 31));
            atomicAdd(&MASK(M_WTOT)[l >> 5], 1u | (static_cast<uint32_t>(wd) << 16));
        }
    }
    __syncthreads();
    {
        const uint32_t nq = min(s.wide_count, static_cast<uint32_t>(kWideQ));
        #pragma unroll 1
        for (uint32_t e = warp; e < nq; e += kWarps) {
            const int l = s.wide_q[e] & 0xffffu, wd = s.wide_q[e] >> 16;
            if (accept_warp(adc_l, noise_l, l, wd, p.tcl2, lane) && lane == 0) {
                atomicOr(&m_acc[l >> 5], 1u << (l & 31));
                atomicAdd(&MASK(M_WTOT)[l >> 5], 1u | (static_cast<uint32_t>(wd) << 16));
            }
        }
    }
    __syncthreads();

    SST_MARK(7);
    // ---------------------------------------------------------------- a7: scan + look-back, warp 0
    // Word totals (accepted clusters | ADC bytes << 16) were accumulated by the accepting lanes.
    // Warp 0 turns them into exclusive prefixes, publishes the FED aggregate and resolves the
    // FED's base offsets with a decoupled look-back over the earlier FEDs.
    uint32_t *const m_wtot = MASK(M_WTOT);
    uint32_t *const m_spre = MASK(M_BRK);  // brk is dead: per-word seed prefix goes here
    const uint32_t fed_over = s.overrun;
    if (warp == 0) {
        const uint32_t K = (nw + 31) >> 5;  // words per lane
        uint32_t my_a = 0, my_s = 0;
        #pragma unroll 1
        for (uint32_t k = 0; k < K; ++k) {
            const uint32_t w = lane * K + k;
            if (w < nw) { my_a += m_wtot[w]; my_s += __popc(m_seed[w]); }
        }
        uint32_t inc_a = my_a, inc_s = my_s;  // FED totals <= 12288 clusters / 24576 ADC bytes: halves stay apart
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t ua = __shfl_up_sync(0xffffffffu, inc_a, d);
            const uint32_t us = __shfl_up_sync(0xffffffffu, inc_s, d);
            if (lane >= d) { inc_a += ua; inc_s += us; }
        }
        const uint32_t tot_a = __shfl_sync(0xffffffffu, inc_a, 31), tot_s = __shfl_sync(0xffffffffu, inc_s, 31);
        const uint32_t fed_cl = tot_a & 0xffffu, fed_adc = tot_a >> 16;
        // publish: word 0 = status | clusters | ADC bytes << 30 (aggregate now, inclusive prefix
        // later); word 1 = ready | seeds | malformed | overrun (aggregate only)
        const unsigned long long agg0 = fed_cl | (static_cast<unsigned long long>(fed_adc) << kShAdc);
        const unsigned long long ep0 = static_cast<unsigned long long>(p.epoch) << kShEp0;
        if (lane == 0) {
            st_state(p.fed_state + 2 * f, (f == 0 ? kStP : kStA) | ep0 | agg0);
            st_state(p.fed_state + 2 * f + 1, kReady | (static_cast<unsigned long long>(p.epoch) << kShEp1) | tot_s |
                                                  (static_cast<unsigned long long>(n_malformed) << kShMalf) |
                                                  (static_cast<unsigned long long>(fed_over) << kShOvr));
        }
        {
            uint32_t ex_a = inc_a - my_a, ex_s = inc_s - my_s;
            #pragma unroll 1
            for (uint32_t k = 0; k < K; ++k) {
                const uint32_t w = lane * K + k;
                if (w < nw) {
                    const uint32_t t = m_wtot[w];
                    m_wtot[w] = ex_a;
                    m_spre[w] = ex_s;
                    ex_a += t;
                    ex_s += __popc(m_seed[w]);
                }
            }
        }
        SST_MARK(8);
        // look-back: lane 0 reads the nearest predecessor; stop at the first inclusive prefix
        unsigned long long excl = 0;
        #pragma unroll 1
        for (int base = static_cast<int>(f) - 1; base >= 0; base -= 32) {
            const int j = base - lane;
            unsigned long long v = kStP;  // before FED 0: prefix 0
            if (j >= 0) {
                v = ld_state(p.fed_state + 2 * j);
                while (!(v >> 62) || ((v >> kShEp0) & 0xffull) != p.epoch) {  // not written by this call yet
                    __nanosleep(64);
                    v = ld_state(p.fed_state + 2 * j);
                }
            }
            const uint32_t pm = __ballot_sync(0xffffffffu, (v >> 62) == 2ull);
            const int stop = pm ? __ffs(pm) - 1 : 31;  // lanes 0..stop contribute
            unsigned long long c = lane <= stop ? (v & kStMask) : 0ull;
#pragma unroll
            for (int o2 = 16; o2 > 0; o2 >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o2);
            excl += c;
            if (pm) break;
        }
        if (lane == 0) {
            if (f) st_state(p.fed_state + 2 * f, kStP | ep0 | (excl + agg0));
            s.red[0][0] = static_cast<uint32_t>(excl & ((1ull << kShAdc) - 1));  // clusters before this FED
            s.red[0][1] = static_cast<uint32_t>(excl >> kShAdc);                 // ADC bytes before this FED
            s.red[0][2] = fed_cl;
            s.red[0][3] = fed_adc;
            s.red[0][4] = tot_s;
        }
    }
    __syncthreads();
    const uint32_t b_cl = s.red[0][0], b_adc = s.red[0][1], fed_cl = s.red[0][2], fed_adc = s.red[0][3],
                   fed_seed = s.red[0][4];

    // seed-index base (only when that output is requested) and, in the last FED, the event totals:
    // sums over the aggregate-only word of every earlier FED
    uint32_t b_seed = 0, b_malf = 0, b_over = 0;
    const bool last = f == p.n_feds - 1;
    if (o.seed_idx || last) {
        #pragma unroll 1
        for (uint32_t j = tid; j < f; j += kThreads) {
            unsigned long long v = ld_state(p.fed_state + 2 * j + 1);
            while (!(v & kReady) || ((v >> kShEp1) & 0xffull) != p.epoch) {
                __nanosleep(100);
                v = ld_state(p.fed_state + 2 * j + 1);
            }
            b_seed += static_cast<uint32_t>(v) & 0xfffffu;
            b_malf += static_cast<uint32_t>(v >> kShMalf) & 0x7fu;
            b_over += static_cast<uint32_t>(v >> kShOvr) & 1u;
        }
        b_seed = warp_sum(b_seed); b_malf = warp_sum(b_malf); b_over = warp_sum(b_over);
        if (lane == 0) { s.red[1][warp] = b_seed; s.red[2][warp] = b_malf; s.red[3][warp] = b_over; }
        __syncthreads();
        b_seed = b_malf = b_over = 0;
#pragma unroll
        for (int i = 0; i < kWarps; ++i) { b_seed += s.red[1][i]; b_malf += s.red[2][i]; b_over += s.red[3][i]; }
    }

    SST_MARK(9);
    // ---------------------------------------------------------------- a7: emit, (module, first strip) order
    if (o.seed_idx) {
        #pragma unroll 1
        for (uint32_t i = tid; i < nw * 32; i += kThreads) {
            const uint32_t w = i >> 5, b = i & 31, sw = m_seed[w];
            if ((sw >> b) & 1u) {
                const uint32_t k = b_seed + m_spre[w] + __popc(sw & ((1u << b) - 1u));
                if (k < o.cap_seeds) o.seed_idx[k] = f * kFedStrips + strip_l[i];
            }
        }
    }
    // ordered list of the FED's accepted clusters (entry | FED-local ADC offset << 16) in the dead
    // run table, then lane per cluster; FEDs with more clusters than the table go in rounds
    uint32_t *const cl_l = s.runs;
    #pragma unroll 1
    for (uint32_t c0 = 0; c0 < fed_cl; c0 += kRunCap) {
        if (c0) __syncthreads();
        #pragma unroll 1
        for (uint32_t w = warp; w < nw; w += kWarps) {
            const uint32_t aw = m_acc[w];
            if (!aw) continue;  // warp-uniform
            const int i = (w << 5) + lane;
            const bool mine = (aw >> lane) & 1u;
            const uint32_t wd = mine ? static_cast<uint32_t>(run_end(m_link, i) - i + 1) : 0u;
            uint32_t incw = wd;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incw, d);
                if (lane >= d) incw += u;
            }
            const uint32_t pre = m_wtot[w];
            const uint32_t c = (pre & 0xffffu) + __popc(aw & ((1u << lane) - 1u)) - c0;
            if (mine && c < static_cast<uint32_t>(kRunCap))
                cl_l[c] = static_cast<uint32_t>(i) | (((pre >> 16) + incw - wd) << 16);
        }
        __syncthreads();
        const uint32_t nc = min(fed_cl - c0, static_cast<uint32_t>(kRunCap));
        #pragma unroll 1
        for (uint32_t c = tid; c < nc; c += kThreads) {
            const uint32_t e = cl_l[c];
            const int i = e & 0xffffu;
            const uint32_t k_cl = b_cl + c0 + c, k_adc = b_adc + (e >> 16);
            const int wd = run_end(m_link, i) - i + 1;
            if (k_cl < o.cap_clusters && k_adc + wd <= o.cap_adc) {
                int Q = 0;
                long long M = 0;
                #pragma unroll 1
                for (int j = 0; j < wd; ++j) {
                    const int q = adc_l[i + j];
                    Q += q;
                    M += static_cast<long long>(j) * q;
                    o.cl_adc[k_adc + j] = static_cast<uint8_t>(q);
                }
                const uint32_t st0 = strip_l[i], ch = st0 >> 8;
                const int first = static_cast<int>(st0) - s.mod_lo[ch] * kStrip;
                o.cl_module[k_cl] = s.mod_id[ch];
                o.cl_first[k_cl] = static_cast<uint16_t>(first);
                o.cl_width[k_cl] = static_cast<uint16_t>(wd);
                o.cl_charge[k_cl] = Q;
                // barycenter in float32: first + M/Q is good to ~2e-7 relative (tolerance 1e-6)
                o.cl_bary[k_cl] = __fadd_rn(static_cast<float>(first),
                                            __fdiv_rn(static_cast<float>(M), static_cast<float>(Q)));
                o.cl_adc_off[k_cl] = k_adc;
                if (o.cl_snr) o.cl_snr[k_cl] = cluster_snr(noise_l, i, wd, Q);
            } else {
                // the first cluster that does not fit reports how many were written
                const bool prev_fits = k_cl == 0 || (k_cl - 1 < o.cap_clusters && k_adc <= o.cap_adc);
                if (prev_fits) *o.n_clusters = k_cl;
            }
        }
    }
    if (last && tid == 0) {  // event totals = prefix of the last FED + its own
        const uint32_t n_cl = b_cl + fed_cl, n_adc = b_adc + fed_adc, n_mal = b_malf + n_malformed,
                       n_over = b_over + fed_over;
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
    SST_MARK(10);
#undef MASK
}

// ------------------------------------------------------------------------------ the kernel
__global__ void __launch_bounds__(kThreads, 5) sst_fed_kernel(const __grid_constant__ KParams p) {
    extern __shared__ __align__(128) uint8_t smem_raw[];
    Smem &s = *reinterpret_cast<Smem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t f = blockIdx.x;
    const sst_output &o = p.out;

    SST_MARK(0);
    // ---------------------------------------------------------------- a1: stage the FED payload
    if (tid == 0) {
        mbar_init(&s.mbar, 1);
        fence_proxy_async();
        const uint32_t fo0 = p.fed_offsets[f], fo1 = p.fed_offsets[f + 1];
        const bool valid = fo0 <= fo1 && fo1 <= p.max_raw_bytes;
        const uint32_t size = valid ? fo1 - fo0 : 0u;
        const bool in_smem = size <= static_cast<uint32_t>(kRawCap) && ((fo0 | size) & 15u) == 0 &&
                             (reinterpret_cast<uintptr_t>(p.raw) & 15u) == 0;
        s.fed_start = fo0;
        s.fed_size = size;
        s.in_smem = in_smem;
        s.overrun = valid ? 0u : 1u;
        s.wide_count = 0;
        s.long_count = 0;
        if (in_smem && size) {
            mbar_expect_tx(&s.mbar, size);
            bulk_g2s(s.u.raw, p.raw + fo0, size, &s.mbar);
        }
    }
    // meanwhile: zero-fill this FED's slice of the dense output, clear the run table, fetch the
    // module map of the 96 channels
    if (o.strip_adc) {
        uint8_t *dst = o.strip_adc + static_cast<size_t>(f) * kFedStrips;
        if ((reinterpret_cast<uintptr_t>(o.strip_adc) & 15u) == 0) {
            uint4 *d4 = reinterpret_cast<uint4 *>(dst);
            const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
            for (int i = 0; i < kFedStrips / 16 / kThreads; ++i) d4[tid + i * kThreads] = z;
        } else {
            #pragma unroll 1
            for (int i = tid; i < kFedStrips; i += kThreads) dst[i] = 0;
        }
    }
    {
        uint4 *r4 = reinterpret_cast<uint4 *>(s.runs);
        const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int i = 0; i < kRunCap / 4 / kThreads; ++i) r4[tid + i * kThreads] = z;
    }
    if (tid < kChan) {
        const uint2 ci = __ldg(p.chan_info + f * kChan + tid);
        s.mod_id[tid] = ci.x;
        s.mod_lo[tid] = static_cast<uint8_t>(ci.y & 0xffu);
        s.mod_hi[tid] = static_cast<uint8_t>((ci.y >> 8) & 0xffu);
    }
    __syncthreads();
    const bool in_smem = s.in_smem != 0;
    const uint32_t fed_size = s.fed_size;
    const uint8_t *rp = in_smem ? s.u.raw : p.raw + s.fed_start;

    SST_MARK(1);
    // ---------------------------------------------------------------- a1: walk the length chain
    if (tid == 0) {
        if (in_smem) {
            if (fed_size) mbar_wait(&s.mbar, 0);
            SST_MARK(2);
            walk_chain_speculative(s.u.raw, s.chan_off, s.chan_len, s.slot_base);
        } else {
            SST_MARK(2);
            if (walk_chain_checked(rp, fed_size, s.overrun != 0, s.chan_off, s.chan_len, s.slot_base)) s.overrun = 1;
        }
    }
    __syncthreads();
    if (in_smem && fed_size) mbar_wait(&s.mbar, 0);  // async-proxy writes visible to every reader
    uint32_t my_off = 0, my_len = 0;
    if (tid < kChan) {
        my_off = s.chan_off[tid];
        my_len = s.chan_len[tid];
    }
    if (in_smem) {  // validate the speculative chain: channels from the first bad one on are empty
        const bool ok = tid >= kChan || (s.overrun == 0 && my_off <= fed_size && my_off + my_len <= fed_size);
        const uint32_t okm = __ballot_sync(0xffffffffu, ok);
        if (lane == 0 && warp < 3) s.okmask[warp] = okm;
        __syncthreads();
        const uint32_t m0 = ~s.okmask[0], m1 = ~s.okmask[1], m2 = ~s.okmask[2];
        const int first_bad = m0 ? __ffs(m0) - 1 : (m1 ? 31 + __ffs(m1) : (m2 ? 63 + __ffs(m2) : kChan));
        if (tid < kChan && tid >= first_bad) {
            my_off = fed_size;
            my_len = 0;
            s.chan_off[tid] = fed_size;
            s.chan_len[tid] = 0;
        }
        if (tid == 0 && first_bad < kChan) s.overrun = 1;
    }
    // the run table is usable if every channel's slot range fits
    const uint32_t n_slots = s.slot_base[kChan];
    const bool table_ok = n_slots <= static_cast<uint32_t>(kRunCap);

    SST_MARK(3);
    // ---------------------------------------------------------------- a2 pass 1: run headers
    // thread per channel: validate the run list, count the strips, fill the run table
    int malformed = 0;
    uint32_t my_cnt = 0;
    if (tid < kChan) {
        if (o.chan_off) o.chan_off[f * kChan + tid] = s.fed_start + my_off;
        if (o.chan_len) o.chan_len[f * kChan + tid] = static_cast<uint16_t>(my_len);
        uint32_t n_runs = 0, n_strips = 0;
        uint32_t *slots = table_ok ? s.runs + s.slot_base[tid] : nullptr;
        const bool ok = in_smem ? scan_runs(s.u.raw, my_off, my_len, tid, slots, n_runs, n_strips)
                                : scan_runs(rp, my_off, my_len, tid, slots, n_runs, n_strips);
        if (ok) {
            my_cnt = n_strips;
        } else {  // a malformed channel contributes no strips
            malformed = 1;
            my_len = 0;
            if (slots)
                #pragma unroll 1
                for (uint32_t k = 0; k < n_runs; ++k) slots[k] = 0;
        }
    }
    // exclusive scan of the 96 counts (warps 0..2)
    uint32_t inc = my_cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += u;
    }
    if (lane == 31 && warp < 3) s.wscan[0][warp] = inc;
    const uint32_t n_malformed = __syncthreads_count(malformed);
    uint32_t my_base = inc - my_cnt;
    if (warp >= 1) my_base += s.wscan[0][0];
    if (warp >= 2) my_base += s.wscan[0][1];
    if (tid < kChan) s.chan_base[tid] = static_cast<uint16_t>(my_base);
    const uint32_t P = s.wscan[0][0] + s.wscan[0][1] + s.wscan[0][2];  // present strips of the FED
    __syncthreads();

    SST_MARK(4);
    if (P <= static_cast<uint32_t>(kListCap))
        lists_to_clusters<true>(p, s, rp, P, table_ok, n_slots, n_malformed, my_off, my_len, my_base);
    else
        lists_to_clusters<false>(p, s, rp, P, table_ok, n_slots, n_malformed, my_off, my_len, my_base);
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
    // per-stream scratch (look-back states + overflow lists), taken from the pool on a stream's
    // first event and kept: stream order makes reuse safe, the epoch makes clearing unnecessary
    struct Slot { cudaStream_t stream; uint8_t *mem; uint32_t epoch; };
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
           o->cl_charge && o->cl_bary && o->cl_adc_off && o->cl_adc;
}

#ifdef SST_PHASE_TIMING
unsigned long long *g_phase_clk = nullptr;
#endif

struct ScratchLayout {
    size_t ents, mwords, o_state, o_noise, o_mask, o_strip, o_adc, total, state_bytes;
};
ScratchLayout scratch_layout(const sst_ctx *ctx) {
    ScratchLayout L{};
    const uint32_t nf = ctx->cfg.n_feds;
    auto up = [](size_t b) { return (b + 255) & ~static_cast<size_t>(255); };
    L.ents = static_cast<size_t>(ctx->cfg.max_raw_bytes) + 16ull * nf + 64;
    L.mwords = L.ents / 32 + 2ull * nf + 16;
    L.state_bytes = 2 * sizeof(unsigned long long) * nf;
    L.o_state = 0;
    L.o_noise = up(L.state_bytes);
    L.o_mask = L.o_noise + up(4 * L.ents);
    L.o_strip = L.o_mask + up(4 * M_COUNT * L.mwords);
    L.o_adc = L.o_strip + up(2 * L.ents);
    L.total = L.o_adc + up(L.ents);
    return L;
}

// The scratch of `st`: allocated (stream-ordered, from the pool) and cleared once, then reused.
sst_status stream_scratch(sst_ctx *ctx, cudaStream_t st, uint8_t **mem, uint32_t *epoch) {
    std::lock_guard<std::mutex> lock(ctx->slot_mu);
    for (auto &sl : ctx->slots)
        if (sl.stream == st) {
            sl.epoch = sl.epoch % 255u + 1u;
            *mem = sl.mem;
            *epoch = sl.epoch;
            return SST_OK;
        }
    const ScratchLayout L = scratch_layout(ctx);
    uint8_t *blk = nullptr;
    SST_CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&blk), L.total, ctx->pool, st));
    SST_CU(cudaMemsetAsync(blk + L.o_state, 0, L.state_bytes, st));
    ctx->slots.push_back({st, blk, 1u});
    *mem = blk;
    *epoch = 1u;
    return SST_OK;
}

sst_status launch_event(sst_ctx *ctx, const uint8_t *raw, const uint32_t *fed_offsets,
                        const sst_thresholds *thr, const sst_output *out, cudaStream_t st) {
    const uint32_t nf = ctx->cfg.n_feds;
    uint8_t *blk = nullptr;
    uint32_t epoch = 0;
    const sst_status rc = stream_scratch(ctx, st, &blk, &epoch);
    if (rc != SST_OK) return rc;
    const ScratchLayout L = scratch_layout(ctx);
    KParams kp{};
    kp.raw = raw;
    kp.fed_offsets = fed_offsets;
    kp.calib = ctx->calib;
    kp.chan_info = ctx->chan_info;
    kp.fed_state = reinterpret_cast<unsigned long long *>(blk + L.o_state);
    kp.g_noise = reinterpret_cast<float *>(blk + L.o_noise);
    kp.g_mask = reinterpret_cast<uint32_t *>(blk + L.o_mask);
    kp.g_mask_words = static_cast<uint32_t>(L.mwords);
    kp.g_strip = reinterpret_cast<uint16_t *>(blk + L.o_strip);
    kp.g_adc = blk + L.o_adc;
    kp.tcl2 = static_cast<double>(thr->cluster) * static_cast<double>(thr->cluster);  // exact
    kp.t_ch = thr->channel;
    kp.t_seed = thr->seed;
    kp.max_raw_bytes = ctx->cfg.max_raw_bytes;
    kp.n_feds = nf;
    kp.epoch = epoch;
    kp.out = *out;
#ifdef SST_PHASE_TIMING
    kp.phase_clk = g_phase_clk;
#endif
    sst_fed_kernel<<<nf, kThreads, sizeof(Smem), st>>>(kp);
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
    if (cudaFuncSetAttribute(sst_fed_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(sizeof(Smem))) != cudaSuccess)
        return fail(SST_ERR_CUDA);
    cudaFuncSetAttribute(sst_fed_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, cfg->device);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctx->ctas_per_sm, sst_fed_kernel, kThreads,
                                                  sizeof(Smem));
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
    if (out->seed_idx == nullptr && out->cap_seeds != 0) return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    return launch_event(ctx, raw, fed_offsets, thr, out, static_cast<cudaStream_t>(stream));
}

sst_status sst_unpack_cluster_batch(sst_ctx *ctx, uint32_t n_events, const uint8_t *const *raw,
                                    const uint32_t *const *fed_offsets, const sst_thresholds *thr,
                                    const sst_output *outs, void *const *streams, uint32_t n_streams) {
    if (!ctx || !raw || !fed_offsets || !thr || !outs || !streams || n_streams == 0 || !thresholds_ok(thr))
        return SST_ERR_INVALID_ARG;
    if (!ctx->has_calib) return SST_ERR_NO_CALIB;
    for (uint32_t e = 0; e < n_events; ++e)
        if (!raw[e] || !fed_offsets[e] || !output_ok(&outs[e]) || (!outs[e].seed_idx && outs[e].cap_seeds))
            return SST_ERR_INVALID_ARG;
    SST_CU(cudaSetDevice(ctx->cfg.device));
    for (uint32_t e = 0; e < n_events; ++e) {
        const sst_status rc = launch_event(ctx, raw[e], fed_offsets[e], thr, &outs[e],
                                           static_cast<cudaStream_t>(streams[e % n_streams]));
        if (rc != SST_OK) return rc;
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
    if (rc == SST_OK) rc = launch_event(ctx, blk + o_raw, reinterpret_cast<uint32_t *>(blk + o_fo), thr, &d, st);
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
    info->smem_bytes = static_cast<uint32_t>(sizeof(Smem));
    info->threads = kThreads;
    info->ctas_per_sm = static_cast<uint32_t>(ctx->ctas_per_sm);
    info->sm_count = static_cast<uint32_t>(ctx->sm_count);
    info->kernels_per_event = 1;
    return SST_OK;
}

}  // extern "C"
