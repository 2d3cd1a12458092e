/*
 * sst_oracle.c -- CPU ORACLE for the strip-tracker unpack + "three thresholds" clustering
 * path of arXiv 2101.11489.
 *
 * THIS IS TEST INFRASTRUCTURE.  It is a plain, sequential, deliberately slow and obviously
 * correct restatement of what the path computes.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or helper with the CUDA path under paper_2101_11489_b200/csrc/.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md; "reading sN" = DESIGN.md section 3):
 *   - raw layout: 96 channels x 256 strips per FED, CSR-like, channel = row, strip = column
 *     (section 2); byte format from BASELINE.json config 0 (readings s1-s3);
 *   - channel-location map, then per-channel unpack into a structure of arrays;
 *   - active strips, seed strips, seed-index array, left/right boundaries, cluster charge,
 *     cluster threshold, outputs (section 2);
 *   - expansion inside a module, one emission per cluster, gain formula, output order and
 *     tolerances: BASELINE.json north_star (readings s4-s18).
 *
 * The method reaches exactly the result of a plain definition, so the clusterer below is
 * that definition written out (not the paper's seed-parallel algorithm):
 *   "within each module the clusters are the maximal runs of contiguous active strips that
 *    contain at least one seed strip and whose charge over quadrature-summed noise reaches
 *    the cluster threshold, listed in ascending strip order".
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"): decode(encode(z)) == z round trip;
 * hand-built byte strings and malformed channels; worked examples W1-W9 with hand-computed
 * expectations (tests/golden/worked_examples.json); exhaustive brute-force interval
 * enumeration on tiny modules (oracle/brute.py, an independent second implementation);
 * runs-of-mask special case against numpy; gain correction against exact rationals;
 * single-strip / equal-noise closed forms for acceptance; invariants and metamorphic checks.
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -shared -fPIC (see sst_oracle.py).
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define SST_O_NCHAN 96
#define SST_O_NSTRIP 256

/* status word bits, same meaning as the library's dev_status[0] (include/sst.h) */
#define SST_O_FLAG_CL_CAP 1u
#define SST_O_FLAG_ADC_CAP 2u
#define SST_O_FLAG_MALFORMED 4u
#define SST_O_FLAG_OVERRUN 8u

/* ---------------------------------------------------------------------------------------
 * Step 1+2: FED walk (channel-location map) and per-channel decode.
 *
 * raw[raw_bytes], fed_offsets[n_feds+1] byte offsets into raw.
 * Outputs: chan_off[n_feds*96] = byte offset of the first run byte of the channel,
 *          chan_len[n_feds*96] = payload length L, adc[n_feds*96*256] dense (absent = 0),
 *          status[0] |= flags, status[1] = malformed channels, status[4] = overrun FEDs.
 * A FED whose offsets are not 0 <= start <= end <= raw_bytes, or whose length chain passes
 * `end`, is flagged; the channel where that happens and all later channels of the FED are
 * empty, recorded as (chan_off = end, chan_len = 0) (reading s3b).  The offsets of an event
 * never step back: a FED whose start lies below an earlier entry of fed_offsets is flagged
 * and empty in the same way (reading s3c), so the FEDs that are decoded never overlap.
 * A malformed channel (reading s2b) contributes no strips.
 * ------------------------------------------------------------------------------------- */
void sst_oracle_unpack(const uint8_t *raw, uint64_t raw_bytes, const uint32_t *fed_offsets,
                       uint32_t n_feds, uint32_t *chan_off, uint16_t *chan_len, uint8_t *adc,
                       uint32_t *status /* [8] */)
{
    uint32_t n_malformed = 0, n_overrun = 0;
    uint64_t fo_max = 0; /* largest of fed_offsets[0..f) */
    for (uint32_t f = 0; f < n_feds; ++f) {
        uint64_t pos = fed_offsets[f];
        uint64_t end = fed_offsets[f + 1];
        int overrun = 0;
        int steps_back = pos < fo_max;
        if (pos > fo_max) fo_max = pos;
        if (steps_back || pos > end || end > raw_bytes) {
            overrun = 1;
            end = pos; /* nothing readable */
        }
        for (uint32_t c = 0; c < SST_O_NCHAN; ++c) {
            uint32_t ch = f * SST_O_NCHAN + c;
            uint8_t *row = adc + (uint64_t)ch * SST_O_NSTRIP;
            memset(row, 0, SST_O_NSTRIP);
            uint64_t off = 0, L = 0;
            if (!overrun) {
                if (pos + 2 > end) {
                    overrun = 1;
                } else {
                    L = (uint64_t)raw[pos] | ((uint64_t)raw[pos + 1] << 8);
                    off = pos + 2;
                    if (off + L > end)
                        overrun = 1;
                }
            }
            if (overrun) {
                chan_off[ch] = (uint32_t)end;
                chan_len[ch] = 0;
                continue;
            }
            chan_off[ch] = (uint32_t)off;
            chan_len[ch] = (uint16_t)L;
            pos = off + L;

            /* decode the runs of this channel into a temporary row; commit only if well formed */
            uint8_t tmp[SST_O_NSTRIP];
            memset(tmp, 0, sizeof tmp);
            uint64_t p = off, pend = off + L;
            uint32_t next_free = 0;
            int ok = 1;
            while (p < pend) {
                if (p + 2 > pend) { ok = 0; break; }
                uint32_t first = raw[p];
                uint32_t len = raw[p + 1];
                if (len == 0) len = 256;                      /* reading s2 */
                if (first < next_free) { ok = 0; break; }     /* overlapping or descending */
                if (first + len > SST_O_NSTRIP) { ok = 0; break; }
                if (p + 2 + len > pend) { ok = 0; break; }    /* run bytes pass the payload */
                for (uint32_t i = 0; i < len; ++i)
                    tmp[first + i] = raw[p + 2 + i];
                next_free = first + len;
                p += 2 + len;
            }
            if (ok)
                memcpy(row, tmp, SST_O_NSTRIP);
            else
                ++n_malformed;
        }
        n_overrun += (uint32_t)overrun;
    }
    status[1] = n_malformed;
    status[4] = n_overrun;
    if (n_malformed) status[0] |= SST_O_FLAG_MALFORMED;
    if (n_overrun) status[0] |= SST_O_FLAG_OVERRUN;
}

/* ---------------------------------------------------------------------------------------
 * Step 3: active / seed flags (readings s4-s9).
 *   active = !bad && adc > 0 && adc/noise >= t_ch      seed = active && adc/noise >= t_seed
 * evaluated exactly: the double product of two float32 values is exact, so
 * (double)adc >= (double)t * (double)noise IS adc/noise >= t in real arithmetic.
 * seed_idx (step "seed-index array") = ascending global ids of seed strips.
 * Returns the number of seeds; seed_idx may be NULL.
 * ------------------------------------------------------------------------------------- */
uint32_t sst_oracle_flags(const uint8_t *adc, const float *noise, const uint8_t *bad, uint64_t n,
                          float t_ch, float t_seed, uint8_t *active, uint8_t *seed,
                          uint32_t *seed_idx)
{
    uint32_t n_seeds = 0;
    for (uint64_t g = 0; g < n; ++g) {
        int a = bad[g] == 0 && adc[g] > 0 &&
                (double)adc[g] >= (double)t_ch * (double)noise[g];
        int s = a && (double)adc[g] >= (double)t_seed * (double)noise[g];
        active[g] = (uint8_t)a;
        seed[g] = (uint8_t)s;
        if (s) {
            if (seed_idx) seed_idx[n_seeds] = (uint32_t)g;
            ++n_seeds;
        }
    }
    return n_seeds;
}

/* Gain correction of one strip (reading s13/s14): float32 RN division, float32 RN add of
 * 0.5f, floor, min with 254.  Exposed so the pins can test it in isolation. */
int32_t sst_oracle_gain_correct(uint8_t adc, float gain)
{
    volatile float t = (float)adc / gain;   /* volatile: no excess precision, no contraction */
    volatile float u = t + 0.5f;
    float fl = floorf(u);
    return fl >= 254.0f ? 254 : (int32_t)fl;   /* min taken before the int conversion */
}

/* ---------------------------------------------------------------------------------------
 * Steps 4+5: per-module sweep and emission (readings s10-s18).
 *
 * Modules are maximal ranges of consecutive channels with equal chan_module[]; they never
 * cross a FED (the caller's map guarantees it; a module id change is also forced at every
 * FED boundary here).  Clusters are emitted in ascending global strip order.
 * Outputs are written up to cap_clusters / cap_adc; counts needed go to status[2], status[3]
 * and the overflow bits to status[0]; *n_clusters = clusters actually written (a prefix).
 * cl_snr (may be NULL) = (float)(Q / sqrt(n2)), for the tolerance check only.
 * ------------------------------------------------------------------------------------- */
void sst_oracle_cluster(const uint8_t *adc, const float *gain, const float *noise,
                        const uint8_t *active, const uint8_t *seed, const uint32_t *chan_module,
                        uint32_t n_feds, float t_cl,
                        uint32_t cap_clusters, uint32_t cap_adc,
                        uint32_t *n_clusters, uint32_t *cl_module, uint16_t *cl_first,
                        uint16_t *cl_width, int32_t *cl_charge, float *cl_bary,
                        uint32_t *cl_adc_off, uint8_t *cl_adc, float *cl_snr,
                        uint32_t *status /* [8] */)
{
    const uint32_t n_chan = n_feds * SST_O_NCHAN;
    uint64_t n_cl = 0, n_adc = 0;   /* needed */
    uint32_t n_written = 0;
    int stopped = 0;                /* once a cluster does not fit nothing later is written */
    const double tcl2 = (double)t_cl * (double)t_cl;   /* exact */

    uint32_t c0 = 0;
    while (c0 < n_chan) {
        uint32_t c1 = c0 + 1;
        while (c1 < n_chan && chan_module[c1] == chan_module[c0] && (c1 % SST_O_NCHAN) != 0)
            ++c1;
        const uint64_t g0 = (uint64_t)c0 * SST_O_NSTRIP, g1 = (uint64_t)c1 * SST_O_NSTRIP;
        uint64_t g = g0;
        while (g < g1) {
            if (!active[g]) { ++g; continue; }
            uint64_t l = g, r = g;
            while (r + 1 < g1 && active[r + 1]) ++r;
            g = r + 1;
            int has_seed = 0;
            for (uint64_t i = l; i <= r; ++i) has_seed |= seed[i];
            if (!has_seed) continue;

            int32_t Q = 0;
            int64_t M = 0;
            double n2 = 0.0;
            for (uint64_t i = l; i <= r; ++i) {
                int32_t q = sst_oracle_gain_correct(adc[i], gain[i]);
                Q += q;
                M += (int64_t)(i - l) * q;
                volatile double sq = (double)noise[i] * (double)noise[i];   /* exact */
                volatile double s = n2 + sq;                               /* one RN add */
                n2 = s;
            }
            volatile double lhs = (double)Q * (double)Q;   /* exact */
            volatile double rhs = tcl2 * n2;               /* one RN multiply */
            if (!(lhs >= rhs)) continue;

            const uint64_t width = r - l + 1;
            if (!stopped && n_cl < cap_clusters && n_adc + width <= cap_adc) {
                const uint32_t k = (uint32_t)n_cl;
                const uint32_t first = (uint32_t)(l - g0);
                cl_module[k] = chan_module[c0];
                cl_first[k] = (uint16_t)first;
                cl_width[k] = (uint16_t)width;
                cl_charge[k] = Q;
                cl_bary[k] = (float)((double)first + (double)M / (double)Q);
                cl_adc_off[k] = (uint32_t)n_adc;
                for (uint64_t i = l; i <= r; ++i)
                    cl_adc[n_adc + (i - l)] = (uint8_t)sst_oracle_gain_correct(adc[i], gain[i]);
                if (cl_snr) cl_snr[k] = (float)((double)Q / sqrt(n2));
                ++n_written;
            } else {
                stopped = 1;
            }
            ++n_cl;
            n_adc += width;
        }
        c0 = c1;
    }
    *n_clusters = n_written;
    status[2] = (uint32_t)n_cl;
    status[3] = (uint32_t)n_adc;
    if (n_cl > cap_clusters) status[0] |= SST_O_FLAG_CL_CAP;
    if (n_adc > cap_adc) status[0] |= SST_O_FLAG_ADC_CAP;
}

/* ---------------------------------------------------------------------------------------
 * Compact structure of arrays: what the paper's unpacker
 * builds -- "unpack the data to SoA format" with "detector conditions (e.g. gain and noise)"
 * per strip, one entry per recorded strip (~800,000 per event).
 * Plain definition: for every global strip id g in ascending order whose dense ADC is non-zero
 * (reading s9: a recorded ADC of 0 carries nothing), the entry (g, adc[g], noise[g], gain[g],
 * bad[g]) with the calibration exactly as it was uploaded.
 * Entries beyond cap are not written; the return value is the number of recorded strips.
 * ------------------------------------------------------------------------------------- */
uint64_t sst_oracle_compact(const uint8_t *adc, const float *gain, const float *noise,
                            const uint8_t *bad, uint64_t n, uint64_t cap, uint32_t *c_strip,
                            uint8_t *c_adc, float *c_noise, float *c_gain, uint8_t *c_bad)
{
    uint64_t k = 0;
    for (uint64_t g = 0; g < n; ++g) {
        if (adc[g] == 0) continue;
        if (k < cap) {
            c_strip[k] = (uint32_t)g;
            c_adc[k] = adc[g];
            c_noise[k] = noise[g];
            c_gain[k] = gain[g];
            c_bad[k] = bad[g] ? 1 : 0;
        }
        ++k;
    }
    return k;
}

/* ---------------------------------------------------------------------------------------
 * Clusters -> global hit coordinates ("convert
 * clusters to global hit coordinates in order to provide the necessary input for MKFIT").
 * The paper gives no geometry; reading s23 fixes a synthetic one: module m is a flat
 * sensor whose strips measure the coordinate u along the direction (-sin phi, cos phi, 0) in
 * the transverse plane, its centre sits at radius r and azimuth phi, at height z:
 *     geom[6 m ..] = { pitch, u0, r, cos phi, sin phi, z }      (float32, as uploaded)
 *     u = u0 + pitch * barycenter            (barycenter in module-local strip units, s16)
 *     x = r cos phi - u sin phi,  y = r sin phi + u cos phi,  z = z
 * evaluated here in double from the float32 inputs and rounded once to float32.
 * A module id >= n_modules gives NaN coordinates.
 * ------------------------------------------------------------------------------------- */
void sst_oracle_hits(const uint32_t *cl_module, const float *cl_bary, uint64_t n_clusters,
                     const float *geom, uint32_t n_modules, float *hit_x, float *hit_y, float *hit_z)
{
    for (uint64_t k = 0; k < n_clusters; ++k) {
        const uint32_t m = cl_module[k];
        if (m >= n_modules) {
            hit_x[k] = hit_y[k] = hit_z[k] = NAN;
            continue;
        }
        const float *gm = geom + 6ull * m;
        const double pitch = gm[0], u0 = gm[1], r = gm[2], c = gm[3], s = gm[4], z = gm[5];
        const double u = u0 + pitch * (double)cl_bary[k];
        hit_x[k] = (float)(r * c - u * s);
        hit_y[k] = (float)(r * s + u * c);
        hit_z[k] = (float)z;
    }
}

