/*
 * sst_oracle_omp.c -- OpenMP TIMING BUILD of the CPU oracle (test infrastructure only).
 *
 * It adds no arithmetic: every strip and cluster is computed by the sequential functions of
 * sst_oracle.c.  It only distributes work in the paper's N x M shape (section 3,
 * Table 1): an outer parallel region over events (N) and an inner one over
 * contiguous FED ranges of one event (M).  Modules never cross a FED, so FED ranges are
 * independent; per-range outputs are concatenated in FED order, which keeps the result
 * bit-identical to the sequential oracle (checked through the hash below by
 * tests/test_oracle_omp.py).  Buffers are allocated and first touched inside the parallel
 * regions ("memory is placed locally to the processor that accesses the data").
 */
#include <omp.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

void sst_oracle_unpack(const uint8_t *raw, uint64_t raw_bytes, const uint32_t *fed_offsets,
                       uint32_t n_feds, uint32_t *chan_off, uint16_t *chan_len, uint8_t *adc,
                       uint32_t *status);
uint32_t sst_oracle_flags(const uint8_t *adc, const float *noise, const uint8_t *bad, uint64_t n,
                          float t_ch, float t_seed, uint8_t *active, uint8_t *seed,
                          uint32_t *seed_idx);
void sst_oracle_cluster(const uint8_t *adc, const float *gain, const float *noise,
                        const uint8_t *active, const uint8_t *seed, const uint32_t *chan_module,
                        uint32_t n_feds, float t_cl, uint32_t cap_clusters, uint32_t cap_adc,
                        uint32_t *n_clusters, uint32_t *cl_module, uint16_t *cl_first,
                        uint16_t *cl_width, int32_t *cl_charge, float *cl_bary,
                        uint32_t *cl_adc_off, uint8_t *cl_adc, float *cl_snr, uint32_t *status);

#define FED_STRIPS (96u * 256u)

/* Work arrays of one FED range (chan_off, chan_len, adc, active, seed): kept per THREAD from call to
 * call and only ever grown, so the timed loop does not pay malloc/free and page faults of ~3 bytes
 * per strip slot per range per event.  Still allocated and first touched by the thread that uses
 * them, inside the parallel region. */
static __thread uint8_t *tl_buf = NULL;
static __thread uint64_t tl_cap = 0;
static uint8_t *thread_work(uint64_t bytes)
{
    if (bytes > tl_cap) {
        free(tl_buf);
        tl_buf = (uint8_t *)malloc(bytes);
        tl_cap = tl_buf ? bytes : 0;
        if (tl_buf) memset(tl_buf, 0, bytes);
    }
    return tl_buf;
}

typedef struct {
    uint32_t n_cl, n_adc, n_seeds;
    uint32_t *cl_module;
    uint16_t *cl_first, *cl_width;
    int32_t *cl_charge;
    float *cl_bary;
    uint32_t *cl_adc_off;
    uint8_t *cl_adc;
} part_t;

static uint64_t fnv(uint64_t h, const void *p, size_t n)
{
    const uint8_t *b = (const uint8_t *)p;
    for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
    return h;
}

/* Processes n_events events; event e has raws[e], raw_bytes[e], fed_offsets[e].  Writes per
 * event the cluster count, the seed count and an FNV-1a hash over the concatenated outputs
 * (module, first, width, charge, bary bits, adc_off per cluster, then all ADC bytes). */
int sst_oracle_events_omp(uint32_t n_events, const uint8_t *const *raws, const uint64_t *raw_bytes,
                          const uint32_t *const *fed_offsets, uint32_t n_feds, const float *gain,
                          const float *noise, const uint8_t *bad, const uint32_t *chan_module,
                          float t_ch, float t_seed, float t_cl, int n_outer, int n_inner,
                          uint32_t *n_clusters_out, uint32_t *n_seeds_out, uint64_t *hash_out)
{
    if (n_outer < 1) n_outer = 1;
    if (n_inner < 1) n_inner = 1;
    if ((uint32_t)n_inner > n_feds) n_inner = (int)n_feds;
    omp_set_max_active_levels(2);
    int failed = 0;
#pragma omp parallel for num_threads(n_outer) schedule(dynamic, 1)
    for (uint32_t e = 0; e < n_events; ++e) {
        part_t *parts = (part_t *)calloc((size_t)n_inner, sizeof(part_t));
#pragma omp parallel for num_threads(n_inner) schedule(static, 1)
        for (int m = 0; m < n_inner; ++m) {
            const uint32_t f0 = (uint32_t)((uint64_t)n_feds * m / n_inner);
            const uint32_t f1 = (uint32_t)((uint64_t)n_feds * (m + 1) / n_inner);
            const uint32_t nf = f1 - f0;
            const uint64_t n = (uint64_t)nf * FED_STRIPS, g0 = (uint64_t)f0 * FED_STRIPS;
            uint32_t status[8] = {0};
            const uint64_t n_al = (n + 63) & ~(uint64_t)63;
            uint8_t *work = thread_work(3 * n_al + (uint64_t)nf * 96 * 6 + 64);
            if (!work) {
#pragma omp atomic write
                failed = 1;
                continue;
            }
            uint8_t *adc = work, *active = work + n_al, *seed = work + 2 * n_al;
            uint32_t *chan_off = (uint32_t *)(work + 3 * n_al);
            uint16_t *chan_len = (uint16_t *)(work + 3 * n_al + (uint64_t)nf * 96 * 4);
            sst_oracle_unpack(raws[e], raw_bytes[e], fed_offsets[e] + f0, nf, chan_off, chan_len,
                              adc, status);
            part_t *p = &parts[m];
            p->n_seeds = sst_oracle_flags(adc, noise + g0, bad + g0, n, t_ch, t_seed, active, seed,
                                          NULL);
            uint32_t cap = 0;
            for (uint64_t i = 0; i < n; ++i) cap += active[i];
            const uint32_t capm = cap ? cap : 1;
            p->cl_module = (uint32_t *)malloc(capm * sizeof(uint32_t));
            p->cl_first = (uint16_t *)malloc(capm * sizeof(uint16_t));
            p->cl_width = (uint16_t *)malloc(capm * sizeof(uint16_t));
            p->cl_charge = (int32_t *)malloc(capm * sizeof(int32_t));
            p->cl_bary = (float *)malloc(capm * sizeof(float));
            p->cl_adc_off = (uint32_t *)malloc(capm * sizeof(uint32_t));
            p->cl_adc = (uint8_t *)malloc(capm);
            sst_oracle_cluster(adc, gain + g0, noise + g0, active, seed, chan_module + f0 * 96, nf,
                               t_cl, cap, cap, &p->n_cl, p->cl_module, p->cl_first, p->cl_width,
                               p->cl_charge, p->cl_bary, p->cl_adc_off, p->cl_adc, NULL, status);
            p->n_adc = status[3];
        }
        /* concatenate in FED order */
        uint64_t h = 14695981039346656037ull;
        uint32_t n_cl = 0, n_adc = 0, n_seeds = 0;
        for (int m = 0; m < n_inner; ++m) {
            part_t *p = &parts[m];
            for (uint32_t k = 0; k < p->n_cl; ++k) {
                uint32_t off = p->cl_adc_off[k] + n_adc;
                h = fnv(h, &p->cl_module[k], 4);
                h = fnv(h, &p->cl_first[k], 2);
                h = fnv(h, &p->cl_width[k], 2);
                h = fnv(h, &p->cl_charge[k], 4);
                h = fnv(h, &p->cl_bary[k], 4);
                h = fnv(h, &off, 4);
            }
            n_cl += p->n_cl;
            n_adc += p->n_adc;
            n_seeds += p->n_seeds;
        }
        for (int m = 0; m < n_inner; ++m) {
            part_t *p = &parts[m];
            h = fnv(h, p->cl_adc, p->n_adc);
            free(p->cl_module); free(p->cl_first); free(p->cl_width); free(p->cl_charge);
            free(p->cl_bary); free(p->cl_adc_off); free(p->cl_adc);
        }
        free(parts);
        n_clusters_out[e] = n_cl;
        n_seeds_out[e] = n_seeds;
        hash_out[e] = h;
    }
    return failed;
}
