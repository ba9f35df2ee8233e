/*
 * Seeded synthetic PairHMM workloads (read x haplotype pairs with per-base qualities).
 *
 * This file holds NO PairHMM arithmetic: it only draws sequences, qualities and pair lists.
 * It serves both the CPU oracle tests and the CUDA path (tests, bench.py) so both see the
 * same bytes.  The shapes follow BASELINE.json configs[0..4] (stand-ins for the paper's GIAB /
 * "10s" data, Table 1 :396-404); the exact recipe is stated in DESIGN.md.
 *
 * Randomness: every item (haplotype, read, region, group) owns a splitmix64 stream seeded by
 * hash(seed, kind, index), so generation is order independent and reproducible.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

typedef struct {
    int64_t n_reads, n_haps, n_pairs;
    int64_t *read_off, *hap_off;                 /* n+1 entries, byte offsets */
    uint8_t *read_bases, *qual_base, *qual_ins, *qual_del, *qual_gcp, *hap_bases;
    int32_t *pair_read, *pair_hap;
} wl_batch;

typedef struct {
    int64_t n;          /* cfg1: regions; cfg2..5: pairs; 0 = default */
    int32_t len_lo;     /* read-length override (0 = default) */
    int32_t len_hi;
} wl_params;

/* ---------------------------------------------------------------- RNG */
typedef struct { uint64_t s; } rng_t;
static inline uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static inline rng_t rng_make(uint64_t seed, uint64_t kind, uint64_t index) {
    rng_t r; r.s = mix64(seed * 0x9E3779B97F4A7C15ULL + mix64(kind * 0xD1B54A32D192ED03ULL + index));
    return r;
}
static inline uint64_t rng_u64(rng_t* r) { r->s += 0x9E3779B97F4A7C15ULL; return mix64(r->s); }
static inline double rng_unif(rng_t* r) { return (double)(rng_u64(r) >> 11) * (1.0 / 9007199254740992.0); }
static inline int64_t rng_int(rng_t* r, int64_t lo, int64_t hi) { /* inclusive */
    return lo + (int64_t)(rng_u64(r) % (uint64_t)(hi - lo + 1));
}
static inline double rng_normal(rng_t* r) {
    double u1 = rng_unif(r), u2 = rng_unif(r);
    if (u1 < 1e-300) u1 = 1e-300;
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
}
static const char ACGT[4] = {'A', 'C', 'G', 'T'};
static inline uint8_t rng_base(rng_t* r) { return (uint8_t)ACGT[rng_u64(r) & 3]; }
static inline uint8_t rng_other_base(rng_t* r, uint8_t b) {
    uint8_t c;
    do { c = rng_base(r); } while (c == b);
    return c;
}
static inline uint8_t qual_normal(rng_t* r, double mu, double sd, int lo, int hi) {
    double v = floor(mu + sd * rng_normal(r) + 0.5);
    if (v < lo) v = lo;
    if (v > hi) v = hi;
    return (uint8_t)v;
}

/* ---------------------------------------------------------------- sequence helpers */
static void fill_random(rng_t* r, uint8_t* dst, int64_t n) { for (int64_t i = 0; i < n; i++) dst[i] = rng_base(r); }

/* Emit exactly `l` bases by walking `src` (length k) from `start` with substitutions and indel
 * events (50/50 insertion/deletion, length uniform 1..indel_max).  If the source is exhausted
 * the remaining bases are uniform random. */
static void mutate_walk(rng_t* r, const uint8_t* src, int64_t k, int64_t start, uint8_t* dst, int64_t l,
                        double sub_rate, double indel_rate, int indel_max) {
    int64_t pos = start, n = 0;
    while (n < l) {
        if (pos >= k) { dst[n++] = rng_base(r); continue; }
        double u = rng_unif(r);
        if (u < indel_rate) {
            int len = (int)rng_int(r, 1, indel_max);
            if (rng_u64(r) & 1) { for (int t = 0; t < len && n < l; t++) dst[n++] = rng_base(r); }
            else pos += len;
            continue;
        }
        uint8_t b = src[pos++];
        if (rng_unif(r) < sub_rate) b = rng_other_base(r, b);
        dst[n++] = b;
    }
}

/* A haplotype of length k derived from a base sequence (length >= k + 16) with n_edits edits
 * (70% SNP, 15% 1-3 bp insertion, 15% 1-3 bp deletion) at uniform positions. */
static void derive_hap(rng_t* r, const uint8_t* base, int64_t base_len, uint8_t* dst, int64_t k, int n_edits) {
    int64_t epos[4]; int etype[4], elen[4];
    for (int e = 0; e < n_edits; e++) {
        epos[e] = rng_int(r, 0, k - 1);
        double u = rng_unif(r);
        etype[e] = u < 0.7 ? 0 : (u < 0.85 ? 1 : 2);
        elen[e] = (int)rng_int(r, 1, 3);
    }
    int64_t pos = 0, n = 0;
    while (n < k) {
        int done = 0;
        for (int e = 0; e < n_edits && !done; e++) {
            if (epos[e] == n && etype[e] >= 0) {
                if (etype[e] == 0) { dst[n++] = rng_other_base(r, base[pos < base_len ? pos : base_len - 1]); pos++; }
                else if (etype[e] == 1) { for (int t = 0; t < elen[e] && n < k; t++) dst[n++] = rng_base(r); }
                else pos += elen[e];
                etype[e] = -1; done = 1;
            }
        }
        if (done) continue;
        dst[n++] = pos < base_len ? base[pos] : rng_base(r);
        pos++;
    }
}

static int alloc_batch(wl_batch* b, int64_t n_reads, int64_t n_haps, int64_t n_pairs) {
    memset(b, 0, sizeof(*b));
    b->n_reads = n_reads; b->n_haps = n_haps; b->n_pairs = n_pairs;
    b->read_off = (int64_t*)calloc((size_t)n_reads + 1, sizeof(int64_t));
    b->hap_off = (int64_t*)calloc((size_t)n_haps + 1, sizeof(int64_t));
    b->pair_read = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_pairs > 0 ? n_pairs : 1));
    b->pair_hap = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_pairs > 0 ? n_pairs : 1));
    return (b->read_off && b->hap_off && b->pair_read && b->pair_hap) ? 0 : -1;
}
static int alloc_payload(wl_batch* b) {
    size_t rb = (size_t)b->read_off[b->n_reads], hb = (size_t)b->hap_off[b->n_haps];
    if (rb == 0) rb = 1;
    if (hb == 0) hb = 1;
    b->read_bases = (uint8_t*)malloc(rb); b->qual_base = (uint8_t*)malloc(rb);
    b->qual_ins = (uint8_t*)malloc(rb); b->qual_del = (uint8_t*)malloc(rb);
    b->qual_gcp = (uint8_t*)malloc(rb); b->hap_bases = (uint8_t*)malloc(hb);
    return (b->read_bases && b->qual_base && b->qual_ins && b->qual_del && b->qual_gcp && b->hap_bases) ? 0 : -1;
}
void wl_free(wl_batch* b) {
    free(b->read_off); free(b->hap_off); free(b->pair_read); free(b->pair_hap);
    free(b->read_bases); free(b->qual_base); free(b->qual_ins); free(b->qual_del); free(b->qual_gcp); free(b->hap_bases);
    memset(b, 0, sizeof(*b));
}

typedef struct { double qb_mu, qb_sd; int qb_lo, qb_hi; double qid_mu, qid_sd; int qid_lo, qid_hi; int gcp; } qual_model;

static void fill_quals(rng_t* r, const wl_batch* b, int64_t read, const qual_model* q) {
    int64_t o = b->read_off[read], l = b->read_off[read + 1] - o;
    for (int64_t i = 0; i < l; i++) {
        b->qual_base[o + i] = qual_normal(r, q->qb_mu, q->qb_sd, q->qb_lo, q->qb_hi);
        if (q->qid_sd > 0) {
            b->qual_ins[o + i] = qual_normal(r, q->qid_mu, q->qid_sd, q->qid_lo, q->qid_hi);
            b->qual_del[o + i] = qual_normal(r, q->qid_mu, q->qid_sd, q->qid_lo, q->qid_hi);
        } else {
            b->qual_ins[o + i] = (uint8_t)q->qid_mu; b->qual_del[o + i] = (uint8_t)q->qid_mu;
        }
        b->qual_gcp[o + i] = (uint8_t)q->gcp;
    }
}

/* ---------------------------------------------------------------- config 0: tiny */
static int gen_cfg0(uint64_t seed, const wl_params* p, wl_batch* b) {
    const int64_t n_reads = 64, n_haps = 4, k = 120, l = p->len_lo > 0 ? p->len_lo : 100;
    if (alloc_batch(b, n_reads, n_haps, n_reads * n_haps)) return -1;
    for (int64_t h = 0; h <= n_haps; h++) b->hap_off[h] = h * k;
    for (int64_t r = 0; r <= n_reads; r++) b->read_off[r] = r * l;
    if (alloc_payload(b)) return -1;
    for (int64_t h = 0; h < n_haps; h++) { rng_t g = rng_make(seed, 1, (uint64_t)h); fill_random(&g, b->hap_bases + h * k, k); }
    qual_model q = {30, 6, 6, 40, 45, 0, 45, 45, 10};
    for (int64_t r = 0; r < n_reads; r++) {
        rng_t g = rng_make(seed, 2, (uint64_t)r);
        int64_t h = rng_int(&g, 0, n_haps - 1);
        int64_t start = rng_int(&g, 0, k - l > 0 ? k - l : 0);
        mutate_walk(&g, b->hap_bases + h * k, k, start, b->read_bases + r * l, l, 0.01, 0.001, 3);
        fill_quals(&g, b, r, &q);
    }
    int64_t n = 0;
    for (int64_t r = 0; r < n_reads; r++) for (int64_t h = 0; h < n_haps; h++) { b->pair_read[n] = (int32_t)r; b->pair_hap[n] = (int32_t)h; n++; }
    return 0;
}

/* ---------------------------------------------------------------- config 1: short-read regions */
static int gen_cfg1(uint64_t seed, const wl_params* p, wl_batch* b) {
    const int64_t n_regions = p->n > 0 ? p->n : 2000, RPR = 128, HPR = 8;
    const int lo = p->len_lo > 0 ? p->len_lo : 100, hi = p->len_hi > 0 ? p->len_hi : 250;
    if (alloc_batch(b, n_regions * RPR, n_regions * HPR, n_regions * RPR * HPR)) return -1;
    int64_t* rlen = (int64_t*)malloc(sizeof(int64_t) * (size_t)n_regions);
    if (!rlen) return -1;
    for (int64_t g = 0; g < n_regions; g++) {
        rng_t r = rng_make(seed, 10, (uint64_t)g);
        rlen[g] = rng_int(&r, lo, hi);
        for (int64_t h = 0; h < HPR; h++) b->hap_off[g * HPR + h + 1] = rlen[g] + rng_int(&r, 20, 250);
        for (int64_t i = 0; i < RPR; i++) b->read_off[g * RPR + i + 1] = rlen[g];
    }
    for (int64_t i = 0; i < b->n_haps; i++) b->hap_off[i + 1] += b->hap_off[i];
    for (int64_t i = 0; i < b->n_reads; i++) b->read_off[i + 1] += b->read_off[i];
    if (alloc_payload(b)) { free(rlen); return -1; }
    qual_model q = {32, 5, 2, 41, 45, 2, 10, 60, 10};
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t g = 0; g < n_regions; g++) {
        uint8_t base[640];
        rng_t r = rng_make(seed, 11, (uint64_t)g);
        fill_random(&r, base, 640);
        for (int64_t h = 0; h < HPR; h++) {
            int64_t hh = g * HPR + h, k = b->hap_off[hh + 1] - b->hap_off[hh];
            rng_t rh = rng_make(seed, 12, (uint64_t)hh);
            derive_hap(&rh, base, 640, b->hap_bases + b->hap_off[hh], k, (int)rng_int(&rh, 0, 3));
        }
        for (int64_t i = 0; i < RPR; i++) {
            int64_t rr = g * RPR + i, l = rlen[g];
            rng_t rd = rng_make(seed, 13, (uint64_t)rr);
            int64_t hh = g * HPR + rng_int(&rd, 0, HPR - 1), k = b->hap_off[hh + 1] - b->hap_off[hh];
            int64_t start = rng_int(&rd, 0, k - l - 8 > 0 ? k - l - 8 : 0);
            mutate_walk(&rd, b->hap_bases + b->hap_off[hh], k, start, b->read_bases + b->read_off[rr], l, 0.01, 0.002, 3);
            fill_quals(&rd, b, rr, &q);
        }
        int64_t n = g * RPR * HPR;
        for (int64_t i = 0; i < RPR; i++) for (int64_t h = 0; h < HPR; h++) {
            b->pair_read[n] = (int32_t)(g * RPR + i); b->pair_hap[n] = (int32_t)(g * HPR + h); n++;
        }
    }
    free(rlen);
    return 0;
}

/* ---------------------------------------------------------------- config 2: mixed-length stream */
static int64_t lognormal_clip(rng_t* r, double median, double sigma, int64_t lo, int64_t hi) {
    double v = floor(median * exp(sigma * rng_normal(r)) + 0.5);
    if (v < (double)lo) v = (double)lo;
    if (v > (double)hi) v = (double)hi;
    return (int64_t)v;
}
static int gen_cfg2(uint64_t seed, const wl_params* p, wl_batch* b) {
    int64_t n_pairs = p->n > 0 ? p->n : 10000000;
    const int64_t RPG = 4, HPG = 2;
    int64_t n_groups = (n_pairs + RPG * HPG - 1) / (RPG * HPG);
    n_pairs = n_groups * RPG * HPG;
    const int lo = p->len_lo > 0 ? p->len_lo : 36, hi = p->len_hi > 0 ? p->len_hi : 300;
    if (alloc_batch(b, n_groups * RPG, n_groups * HPG, n_pairs)) return -1;
    for (int64_t g = 0; g < n_groups; g++) {
        rng_t r = rng_make(seed, 20, (uint64_t)g);
        int64_t maxl = 0;
        for (int64_t i = 0; i < RPG; i++) {
            int64_t l = lognormal_clip(&r, 150, 0.35, lo, hi);
            b->read_off[g * RPG + i + 1] = l;
            if (l > maxl) maxl = l;
        }
        for (int64_t h = 0; h < HPG; h++) {
            int64_t k;
            do { k = lognormal_clip(&r, 350, 0.45, 40, 1200); } while (k < maxl + 10);
            b->hap_off[g * HPG + h + 1] = k;
        }
    }
    for (int64_t i = 0; i < b->n_haps; i++) b->hap_off[i + 1] += b->hap_off[i];
    for (int64_t i = 0; i < b->n_reads; i++) b->read_off[i + 1] += b->read_off[i];
    if (alloc_payload(b)) return -1;
    qual_model q = {32, 5, 2, 41, 45, 2, 10, 60, 10};
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t g = 0; g < n_groups; g++) {
        uint8_t base[1232];
        rng_t r = rng_make(seed, 21, (uint64_t)g);
        fill_random(&r, base, 1232);
        for (int64_t h = 0; h < HPG; h++) {
            int64_t hh = g * HPG + h, k = b->hap_off[hh + 1] - b->hap_off[hh];
            rng_t rh = rng_make(seed, 22, (uint64_t)hh);
            derive_hap(&rh, base, 1232, b->hap_bases + b->hap_off[hh], k, (int)rng_int(&rh, 0, 3));
        }
        for (int64_t i = 0; i < RPG; i++) {
            int64_t rr = g * RPG + i, l = b->read_off[rr + 1] - b->read_off[rr];
            rng_t rd = rng_make(seed, 23, (uint64_t)rr);
            if (rng_unif(&rd) < 0.05) {
                fill_random(&rd, b->read_bases + b->read_off[rr], l);        /* unrelated read */
            } else {
                int64_t hh = g * HPG + rng_int(&rd, 0, HPG - 1), k = b->hap_off[hh + 1] - b->hap_off[hh];
                int64_t start = rng_int(&rd, 0, k - l - 8 > 0 ? k - l - 8 : 0);
                mutate_walk(&rd, b->hap_bases + b->hap_off[hh], k, start, b->read_bases + b->read_off[rr], l, 0.01, 0.002, 3);
            }
            fill_quals(&rd, b, rr, &q);
        }
        int64_t n = g * RPG * HPG;
        for (int64_t i = 0; i < RPG; i++) for (int64_t h = 0; h < HPG; h++) {
            b->pair_read[n] = (int32_t)(g * RPG + i); b->pair_hap[n] = (int32_t)(g * HPG + h); n++;
        }
    }
    /* global Fisher-Yates shuffle of the pair list: the stream arrives unsorted */
    rng_t s = rng_make(seed, 24, 0);
    for (int64_t i = n_pairs - 1; i > 0; i--) {
        int64_t j = (int64_t)(rng_u64(&s) % (uint64_t)(i + 1));
        int32_t t = b->pair_read[i]; b->pair_read[i] = b->pair_read[j]; b->pair_read[j] = t;
        t = b->pair_hap[i]; b->pair_hap[i] = b->pair_hap[j]; b->pair_hap[j] = t;
    }
    return 0;
}

/* ---------------------------------------------------------------- configs 3/4: long reads; 5: equal-length sweep */
static int gen_long(uint64_t seed, const wl_params* p, wl_batch* b, int cfg) {
    int64_t n_pairs = p->n > 0 ? p->n : (cfg == 3 ? 2000 : 16);
    int64_t lo = cfg == 3 ? 5000 : 100000, hi = cfg == 3 ? 15000 : 100000;
    if (p->len_lo > 0) { lo = p->len_lo; hi = p->len_hi > 0 ? p->len_hi : p->len_lo; }
    if (alloc_batch(b, n_pairs, n_pairs, n_pairs)) return -1;
    for (int64_t i = 0; i < n_pairs; i++) {
        rng_t r = rng_make(seed, 30, (uint64_t)i);
        int64_t l = rng_int(&r, lo, hi);
        int64_t k = cfg == 3 ? (int64_t)floor((double)l * (1.05 + 0.15 * rng_unif(&r)) + 0.5)
                             : (int64_t)floor((double)l * 1.05 + 0.5);
        b->read_off[i + 1] = l; b->hap_off[i + 1] = k;
        b->pair_read[i] = (int32_t)i; b->pair_hap[i] = (int32_t)i;
    }
    for (int64_t i = 0; i < n_pairs; i++) { b->hap_off[i + 1] += b->hap_off[i]; b->read_off[i + 1] += b->read_off[i]; }
    if (alloc_payload(b)) return -1;
    qual_model q = {20, 6, 3, 40, 25, 5, 5, 60, 10};
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n_pairs; i++) {
        int64_t l = b->read_off[i + 1] - b->read_off[i], k = b->hap_off[i + 1] - b->hap_off[i];
        rng_t rh = rng_make(seed, 31, (uint64_t)i);
        fill_random(&rh, b->hap_bases + b->hap_off[i], k);
        rng_t rd = rng_make(seed, 32, (uint64_t)i);
        int64_t start = rng_int(&rd, 0, k - l > 0 ? k - l : 0);
        mutate_walk(&rd, b->hap_bases + b->hap_off[i], k, start, b->read_bases + b->read_off[i], l, 0.05, 0.03, 5);
        fill_quals(&rd, b, i, &q);
    }
    return 0;
}
/* cfg 5: the paper's scalability-sweep shape: n pairs, read length = haplotype
 * length = len_lo, read = noisy copy of the haplotype (config-1 error model and quals). */
static int gen_equal(uint64_t seed, const wl_params* p, wl_batch* b) {
    int64_t n_pairs = p->n > 0 ? p->n : 1024, L = p->len_lo > 0 ? p->len_lo : 512;
    if (alloc_batch(b, n_pairs, n_pairs, n_pairs)) return -1;
    for (int64_t i = 0; i < n_pairs; i++) {
        b->read_off[i + 1] = (i + 1) * L; b->hap_off[i + 1] = (i + 1) * L;
        b->pair_read[i] = (int32_t)i; b->pair_hap[i] = (int32_t)i;
    }
    if (alloc_payload(b)) return -1;
    qual_model q = {32, 5, 2, 41, 45, 2, 10, 60, 10};
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n_pairs; i++) {
        rng_t rh = rng_make(seed, 51, (uint64_t)i);
        fill_random(&rh, b->hap_bases + i * L, L);
        rng_t rd = rng_make(seed, 52, (uint64_t)i);
        mutate_walk(&rd, b->hap_bases + i * L, L, 0, b->read_bases + i * L, L, 0.01, 0.002, 3);
        fill_quals(&rd, b, i, &q);
    }
    return 0;
}

int wl_generate(int cfg, uint64_t seed, const wl_params* params, wl_batch* out) {
    wl_params p; memset(&p, 0, sizeof(p));
    if (params) p = *params;
    int rc;
    switch (cfg) {
        case 0: rc = gen_cfg0(seed, &p, out); break;
        case 1: rc = gen_cfg1(seed, &p, out); break;
        case 2: rc = gen_cfg2(seed, &p, out); break;
        case 3: case 4: rc = gen_long(seed, &p, out, cfg); break;
        case 5: rc = gen_equal(seed, &p, out); break;
        default: return -2;
    }
    if (rc) wl_free(out);
    return rc;
}
