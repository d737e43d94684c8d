/*
 * asr_oracle.c -- CPU ORACLE (test infrastructure, NOT the product).
 * See asr_oracle.h for the rules that govern this directory.
 *
 * Every function follows the passage it cites, in the paper's order, with no
 * blocking, fusion or fast-forwarding: the simulator steps ONE engine
 * iteration at a time and the selector is "sort everything, take k".
 */
#define _GNU_SOURCE
#include "asr_oracle.h"

#include <stdlib.h>
#include <string.h>

typedef __int128 i128;

/* ------------------------------------------------------------------ */
/* c1. comparator (readings S2-S6)                           */
/* ------------------------------------------------------------------ */

static int64_t est_of(const orc_req_t *r) {
    /* PAPER.md:260  estimated_output = max(1, int(duration_s * kappa)) */
    return r->est < 1 ? 1 : (int64_t)r->est;
}

static int64_t wait_of(const orc_req_t *r, int64_t now) {
    /* PAPER.md:281  wait = now - req.arrival_time (never negative here) */
    int64_t w = now - r->arrival_us;
    return w < 0 ? 0 : w;
}

/* (arrival_us, idx) ascending: FCFS and every tie-break */
static int earlier(const orc_req_t *a, int64_t ia, const orc_req_t *b,
                   int64_t ib) {
    if (a->arrival_us != b->arrival_us) return a->arrival_us < b->arrival_us;
    return ia < ib;
}

/* "The oracle multiplies in __int128 and asserts the products
 * fit int64".  The boundary's documented bound is wait * est < 2^62
 * (wait < 2^38, est <= 2^24).  A product at or beyond it is counted here and
 * turned into error -4 by orc_select / orc_simulate* / orc_itl, so an input
 * outside the boundary's contract is caught by the checker instead of being
 * compared against an int64 path that may have wrapped.  The ordering itself
 * stays exact in 128 bits. */
static __thread int64_t g_bound_violations = 0;
static const i128 HRRN_PRODUCT_BOUND = (i128)1 << 62;

int64_t orc_bound_violations(void) { return g_bound_violations; }
void orc_bound_violations_reset(void) { g_bound_violations = 0; }

int orc_better(const orc_req_t *a, int64_t ia, const orc_req_t *b, int64_t ib,
               int policy, int64_t now) {
    if (policy == ORC_FCFS) return earlier(a, ia, b, ib);
    if (policy == ORC_SJF) {
        /* PAPER.md:270,277 key (estimated_output_tokens, arrival_time,
         * request_id); "earlier arrivals are prioritized" */
        int64_t ea = est_of(a), eb = est_of(b);
        if (ea != eb) return ea < eb;
        return earlier(a, ia, b, ib);
    }
    /* HRRN: ratio (wait + est) / est, highest first.
     * (wa+ea)/ea > (wb+eb)/eb  <=>  wa*eb > wb*ea   (all positive),
     * evaluated exactly in 128-bit integers. */
    i128 lhs = (i128)wait_of(a, now) * (i128)est_of(b);
    i128 rhs = (i128)wait_of(b, now) * (i128)est_of(a);
    if (lhs >= HRRN_PRODUCT_BOUND || rhs >= HRRN_PRODUCT_BOUND) g_bound_violations++;
    if (lhs != rhs) return lhs > rhs;
    return earlier(a, ia, b, ib);
}

typedef struct {
    const orc_req_t *q;
    int policy;
    int64_t now;
} sort_ctx_t;

static int cmp_pos(const void *pa, const void *pb, void *vctx) {
    const sort_ctx_t *c = (const sort_ctx_t *)vctx;
    int64_t ia = *(const int64_t *)pa, ib = *(const int64_t *)pb;
    if (ia == ib) return 0;
    return orc_better(&c->q[ia], ia, &c->q[ib], ib, c->policy, c->now) ? -1 : 1;
}

/* Select = sort all n positions by the total order, output the first k. */
int orc_select(const orc_req_t *q, int64_t n, int policy, int64_t now,
               int32_t k, int32_t *out_idx) {
    if (n < 0 || k < 0 || policy < 0 || policy > 2) return -1;
    int64_t *pos = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
    if (!pos) return -2;
    for (int64_t i = 0; i < n; i++) pos[i] = i;
    sort_ctx_t c = {q, policy, now};
    const int64_t v0 = g_bound_violations;
    qsort_r(pos, (size_t)n, sizeof(int64_t), cmp_pos, &c);
    for (int32_t j = 0; j < k; j++) out_idx[j] = j < n ? (int32_t)pos[j] : -1;
    free(pos);
    return g_bound_violations != v0 ? -4 : 0;
}

/* ------------------------------------------------------------------ */
/* c2. simulator                                                       */
/* ------------------------------------------------------------------ */

int64_t orc_tokens(const orc_cost_t *cm, int32_t dur_ms) {
    /* BASELINE.json configs[0]: tokens = 1 + 4*dur_ms/1000 (floor);
     * 5 tokens per second of audio in the toy */
    int64_t t = (int64_t)cm->tok_base +
                ((int64_t)cm->tok_per_s * (int64_t)dur_ms) / 1000;
    return t < 1 ? 1 : t;
}

int64_t orc_enc_cost(const orc_cost_t *cm, int32_t dur_ms) {
    /* PAPER.md:51 near-constant encoder time per segment (+ linear term of
     * BASELINE.json configs[0]: 20,000 + 2*dur_ms us) */
    return cm->enc_base_us + cm->enc_per_ms_us * (int64_t)dur_ms;
}

/* order the waiting positions by the total order, at one fixed `now` */
typedef struct {
    const orc_req_t *trace;
    int policy;
    int64_t now;
} wait_ctx_t;

static int cmp_wait(const void *pa, const void *pb, void *vctx) {
    const wait_ctx_t *c = (const wait_ctx_t *)vctx;
    int64_t ia = *(const int64_t *)pa, ib = *(const int64_t *)pb;
    if (ia == ib) return 0;
    return orc_better(&c->trace[ia], ia, &c->trace[ib], ib, c->policy, c->now)
               ? -1
               : 1;
}

int orc_simulate(const orc_req_t *trace, int64_t n, int policy,
                 const orc_cost_t *cm, int32_t slots, int64_t *lat,
                 int64_t *ttft, int64_t *first_arrival_us,
                 int64_t *last_done_us) {
    if (n < 0 || slots < 1 || policy < 0 || policy > 2 || !cm) return -1;
    if (first_arrival_us) *first_arrival_us = n > 0 ? trace[0].arrival_us : 0;
    if (last_done_us) *last_done_us = 0;
    if (n == 0) return 0;

    int64_t *W = (int64_t *)malloc(sizeof(int64_t) * (size_t)n); /* waiting */
    int64_t *R = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots); /* running idx */
    int64_t *rem = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots);
    if (!W || !R || !rem) {
        free(W); free(R); free(rem);
        return -2;
    }
    int64_t nW = 0, nR = 0, p = 0, done = 0, t = 0;
    const int64_t v0 = g_bound_violations;

    while (done < n) {
        /* 1. ingest: arrivals at or before the iteration boundary (S13) */
        while (p < n && trace[p].arrival_us <= t) W[nW++] = p++;
        /* 2. idle server: clock jumps exactly to the next arrival (S14) */
        if (nR == 0 && nW == 0) {
            t = trace[p].arrival_us;
            continue;
        }
        /* 3. admit the k best waiting requests into the free slots (S6:
         *    one `now` = t for the whole step) */
        int64_t free_slots = (int64_t)slots - nR;
        int64_t k = free_slots < nW ? free_slots : nW;
        int64_t enc_sum = 0;
        int64_t first_new = nR;
        if (k > 0) {
            wait_ctx_t c = {trace, policy, t};
            qsort_r(W, (size_t)nW, sizeof(int64_t), cmp_wait, &c);
            for (int64_t j = 0; j < k; j++) {
                int64_t i = W[j];
                R[nR] = i;
                rem[nR] = orc_tokens(cm, trace[i].dur_ms);
                nR++;
                enc_sum += orc_enc_cost(cm, trace[i].dur_ms); /* S15 */
            }
            memmove(W, W + k, sizeof(int64_t) * (size_t)(nW - k));
            nW -= k;
        }
        /* 4. one engine iteration (PAPER.md:31 iteration-level scheduling):
         *    encoders of the admitted + one decode step for everyone (S16) */
        t += enc_sum + cm->iter_base_us + cm->iter_per_running_us * nR;
        for (int64_t s = 0; s < nR; s++) rem[s] -= 1;
        /* 5. record: first token of the admitted (S9), finished requests */
        for (int64_t s = first_new; s < nR; s++)
            ttft[R[s]] = t - trace[R[s]].arrival_us;
        int64_t keep = 0;
        for (int64_t s = 0; s < nR; s++) {
            if (rem[s] == 0) {
                lat[R[s]] = t - trace[R[s]].arrival_us; /* PAPER.md:100 E2EL */
                done++;
            } else {
                R[keep] = R[s];
                rem[keep] = rem[s];
                keep++;
            }
        }
        nR = keep;
    }
    if (last_done_us) *last_done_us = t;
    free(W); free(R); free(rem);
    return g_bound_violations != v0 ? -4 : 0;
}

/* ------------------------------------------------------------------ */
/* 8(f) extensions: preemption, policy switching           */
/* (PAPER.md:156), TPOT, estimator          */
/* ------------------------------------------------------------------ */

static int eff_policy(int policy, const orc_ext_t *ext, int64_t n_waiting) {
    if (policy != ORC_ADAPTIVE) return policy;
    if (n_waiting < ext->depth1) return ext->pol[0];
    if (n_waiting < ext->depth2) return ext->pol[1];
    return ext->pol[2];
}

static int64_t kv_enc(const orc_ext_t *ext, int32_t dur_ms) {
    return ext->kv_base + (ext->kv_per_s * (int64_t)dur_ms) / 1000;
}

int orc_simulate_ex(const orc_req_t *trace, int64_t n, int policy,
                    const orc_cost_t *cm, const orc_ext_t *ext, int32_t slots,
                    int64_t *lat, int64_t *ttft, int64_t *first_arrival_us,
                    int64_t *last_done_us, int64_t *n_preempt) {
    if (n_preempt) *n_preempt = 0;
    if (!ext) {
        if (policy == ORC_ADAPTIVE) return -1;
        return orc_simulate(trace, n, policy, cm, slots, lat, ttft,
                            first_arrival_us, last_done_us);
    }
    if (n < 0 || slots < 1 || policy < 0 || policy > 3 || !cm) return -1;
    if (policy == ORC_ADAPTIVE) {
        if (ext->depth1 > ext->depth2) return -1;
        for (int j = 0; j < 3; j++)
            if (ext->pol[j] < 0 || ext->pol[j] > 2) return -1;
    }
    const int64_t B = ext->kv_budget;
    if (B > 0) /* E8: every request must fit alone, or it could never finish */
        for (int64_t i = 0; i < n; i++)
            if (kv_enc(ext, trace[i].dur_ms) + orc_tokens(cm, trace[i].dur_ms) > B)
                return -3;
    if (first_arrival_us) *first_arrival_us = n > 0 ? trace[0].arrival_us : 0;
    if (last_done_us) *last_done_us = 0;
    if (n == 0) return 0;

    int64_t *W = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    int64_t *R = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots);
    int64_t *rem = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots);
    int64_t *mem = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots);
    char *fresh = (char *)malloc((size_t)slots);      /* admitted in this step */
    char *ever = (char *)calloc((size_t)n, 1);        /* had a first token */
    if (!W || !R || !rem || !mem || !fresh || !ever) {
        free(W); free(R); free(rem); free(mem); free(fresh); free(ever);
        return -2;
    }
    int64_t nW = 0, nR = 0, p = 0, done = 0, t = 0;
    int blocked = 0; /* E6: admission cut short by memory; retried only
                        after the waiting or the running set has changed */
    const int64_t v0 = g_bound_violations;

    while (done < n) {
        /* 1. ingest (S13) */
        while (p < n && trace[p].arrival_us <= t) {
            W[nW++] = p++;
            blocked = 0;
        }
        /* 2. idle server (S14) */
        if (nR == 0 && nW == 0) {
            t = trace[p].arrival_us;
            continue;
        }
        const int pol = eff_policy(policy, ext, nW); /* E7: depth after ingest */
        /* 3a. memory pressure (E1-E4): one more token for everyone must fit */
        int64_t preempted = 0;
        if (B > 0) {
            int64_t M = 0;
            for (int64_t s = 0; s < nR; s++) M += mem[s];
            while (M + nR > B) { /* nR >= 2 here by E8 */
                int64_t v = 0;   /* the WORST running request at now = t */
                for (int64_t s = 1; s < nR; s++)
                    if (orc_better(&trace[R[v]], R[v], &trace[R[s]], R[s], pol, t))
                        v = s;
                W[nW++] = R[v]; /* waits again, keeps its arrival time */
                M -= mem[v];
                for (int64_t s = v + 1; s < nR; s++) {
                    R[s - 1] = R[s];
                    rem[s - 1] = rem[s];
                    mem[s - 1] = mem[s];
                }
                nR--;
                preempted++;
                blocked = 0;
            }
        }
        if (n_preempt) *n_preempt += preempted;
        /* 3b. admission: only in a step without preemption (E5) */
        int64_t enc_sum = 0;
        for (int64_t s = 0; s < nR; s++) fresh[s] = 0;
        if (preempted == 0 && !blocked && nW > 0 && nR < slots) {
            wait_ctx_t c = {trace, pol, t};
            qsort_r(W, (size_t)nW, sizeof(int64_t), cmp_wait, &c);
            int64_t M = 0;
            for (int64_t s = 0; s < nR; s++) M += mem[s];
            int64_t k = 0;
            while (k < nW && nR < slots) {
                int64_t i = W[k];
                int64_t kv = B > 0 ? kv_enc(ext, trace[i].dur_ms) : 0;
                if (B > 0 && M + kv + nR + 1 > B) { /* head of line does not fit */
                    blocked = 1;
                    break;
                }
                R[nR] = i;
                rem[nR] = orc_tokens(cm, trace[i].dur_ms);
                mem[nR] = kv;
                fresh[nR] = 1;
                M += kv;
                nR++;
                k++;
                enc_sum += orc_enc_cost(cm, trace[i].dur_ms); /* recompute pays again */
            }
            memmove(W, W + k, sizeof(int64_t) * (size_t)(nW - k));
            nW -= k;
        }
        /* 4. one engine iteration */
        t += enc_sum + cm->iter_base_us + cm->iter_per_running_us * nR;
        for (int64_t s = 0; s < nR; s++) {
            rem[s] -= 1;
            mem[s] += 1;
        }
        /* 5. record */
        for (int64_t s = 0; s < nR; s++)
            if (fresh[s] && !ever[R[s]]) {
                ttft[R[s]] = t - trace[R[s]].arrival_us; /* first admission only */
                ever[R[s]] = 1;
            }
        int64_t keep = 0;
        for (int64_t s = 0; s < nR; s++) {
            if (rem[s] == 0) {
                lat[R[s]] = t - trace[R[s]].arrival_us;
                done++;
                blocked = 0;
            } else {
                R[keep] = R[s];
                rem[keep] = rem[s];
                mem[keep] = mem[s];
                keep++;
            }
        }
        nR = keep;
    }
    if (last_done_us) *last_done_us = t;
    free(W); free(R); free(rem); free(mem); free(fresh); free(ever);
    return g_bound_violations != v0 ? -4 : 0;
}

int orc_itl(const orc_req_t *trace, int64_t n, int policy, const orc_cost_t *cm,
            int32_t slots, const int32_t *pcts, int32_t n_pct, int64_t *out_pcts,
            int64_t *out_count, int64_t *out_sum) {
    if (n < 0 || slots < 1 || policy < 0 || policy > 2 || !cm || n_pct < 0) return -1;
    int64_t cap = 1024, cnt = 0, sum = 0;
    int64_t *gaps = (int64_t *)malloc(sizeof(int64_t) * (size_t)cap);
    int64_t *W = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
    int64_t *R = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots);
    int64_t *rem = (int64_t *)malloc(sizeof(int64_t) * (size_t)slots);
    if (!gaps || !W || !R || !rem) {
        free(gaps); free(W); free(R); free(rem);
        return -2;
    }
    int64_t nW = 0, nR = 0, p = 0, done = 0, t = 0;
    const int64_t v0 = g_bound_violations;
    while (done < n) { /* the loop of orc_simulate, one iteration at a time */
        while (p < n && trace[p].arrival_us <= t) W[nW++] = p++;
        if (nR == 0 && nW == 0) {
            t = trace[p].arrival_us;
            continue;
        }
        int64_t free_slots = (int64_t)slots - nR;
        int64_t k = free_slots < nW ? free_slots : nW;
        int64_t enc_sum = 0, already = nR;
        if (k > 0) {
            wait_ctx_t c = {trace, policy, t};
            qsort_r(W, (size_t)nW, sizeof(int64_t), cmp_wait, &c);
            for (int64_t j = 0; j < k; j++) {
                int64_t i = W[j];
                R[nR] = i;
                rem[nR] = orc_tokens(cm, trace[i].dur_ms);
                nR++;
                enc_sum += orc_enc_cost(cm, trace[i].dur_ms);
            }
            memmove(W, W + k, sizeof(int64_t) * (size_t)(nW - k));
            nW -= k;
        }
        const int64_t dt = enc_sum + cm->iter_base_us + cm->iter_per_running_us * nR;
        t += dt;
        for (int64_t s = 0; s < already; s++) { /* one gap per request that was running */
            if (cnt == cap) {
                cap *= 2;
                int64_t *g2 = (int64_t *)realloc(gaps, sizeof(int64_t) * (size_t)cap);
                if (!g2) {
                    free(gaps); free(W); free(R); free(rem);
                    return -2;
                }
                gaps = g2;
            }
            gaps[cnt++] = dt;
            sum += dt;
        }
        int64_t keep = 0;
        for (int64_t s = 0; s < nR; s++) {
            rem[s] -= 1;
            if (rem[s] == 0) {
                done++;
            } else {
                R[keep] = R[s];
                rem[keep] = rem[s];
                keep++;
            }
        }
        nR = keep;
    }
    for (int32_t j = 0; j < n_pct; j++) out_pcts[j] = orc_percentile(gaps, cnt, pcts[j]);
    if (out_count) *out_count = cnt;
    if (out_sum) *out_sum = sum;
    free(gaps); free(W); free(R); free(rem);
    return g_bound_violations != v0 ? -4 : 0;
}

int orc_tpot(const orc_req_t *trace, int64_t n, const orc_cost_t *cm,
             const int64_t *lat, const int64_t *ttft, int64_t *out) {
    if (n < 0 || !cm) return -1;
    for (int64_t i = 0; i < n; i++) {
        int64_t tok = orc_tokens(cm, trace[i].dur_ms);
        out[i] = tok > 1 ? (lat[i] - ttft[i]) / (tok - 1) : -1;
    }
    return 0;
}

int orc_estimate(orc_req_t *recs, int64_t n, const int32_t *kappa_milli_by_lang,
                 int32_t n_lang, const uint8_t *lang, const int32_t *speech_ms) {
    if (n < 0 || n_lang < 1 || !kappa_milli_by_lang) return -1;
    for (int64_t i = 0; i < n; i++) {
        int32_t l = lang ? (int32_t)lang[i] : 0;
        if (l >= n_lang) l = 0; /* DESIGN.md reading E12: an unknown language id uses entry 0 */
        int64_t d = speech_ms ? speech_ms[i] : recs[i].dur_ms;
        if (d < 0) d = 0;
        int64_t e = (d * (int64_t)kappa_milli_by_lang[l]) / 1000000;
        if (e < 1) e = 1;
        if (e > ((int64_t)1 << 24)) e = (int64_t)1 << 24; /* DESIGN.md reading E10: the
                                        comparator's documented bound est <= 2^24 */
        recs[i].est = (int32_t)e;
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* c3. nearest-rank percentile (S8)            */
/* ------------------------------------------------------------------ */

static int cmp_i64(const void *a, const void *b) {
    int64_t x = *(const int64_t *)a, y = *(const int64_t *)b;
    return (x > y) - (x < y);
}

int64_t orc_percentile(const int64_t *v, int64_t n, int32_t p) {
    if (n <= 0 || p < 1 || p > 100) return -1;
    int64_t *s = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    if (!s) return -1;
    memcpy(s, v, sizeof(int64_t) * (size_t)n);
    qsort(s, (size_t)n, sizeof(int64_t), cmp_i64);
    /* 1-based rank ceil(p*n/100) */
    int64_t rank = ((int64_t)p * n + 99) / 100;
    int64_t r = s[rank - 1];
    free(s);
    return r;
}

/* ------------------------------------------------------------------ */
/* c4. counter-based trace generator        */
/* ------------------------------------------------------------------ */

uint64_t orc_fmix64(uint64_t z) {
    /* the output function of splitmix64 (Steele, Lea, Flood 2014) */
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t orc_mix64(uint64_t seed, uint32_t stream, uint64_t i) {
    /* a splitmix64 stream whose start state is a hash of (seed, stream);
     * draw i is the (i+1)-th output of that stream */
    uint64_t base = orc_fmix64(orc_fmix64(seed + 0x2545F4914F6CDD1DULL) +
                               (uint64_t)stream * 0xD1B54A32D192ED03ULL);
    return orc_fmix64(base + (i + 1) * 0x9E3779B97F4A7C15ULL);
}

/* T[hi] + ((T[hi+1]-T[hi]) * fr >> 32): 12-bit cell, 32-bit fraction */
static uint64_t interp_tab(const uint32_t *T, uint64_t u) {
    uint64_t hi = u >> 52;
    uint64_t fr = (u >> 20) & 0xFFFFFFFFULL;
    uint64_t lo_v = T[hi], hi_v = T[hi + 1];
    return lo_v + (((hi_v - lo_v) * fr) >> 32);
}

static int clz64(uint64_t x) { /* x != 0 */
    int c = 0;
    while (!(x >> 63)) {
        x <<= 1;
        c++;
    }
    return c;
}

static int32_t draw_duration(uint64_t u, int32_t dist, const uint32_t *ln_dur) {
    if (dist == ORC_DIST_UNIFORM) /* integer ms, uniform on [1000, 35000] */
        return (int32_t)(1000 + (((u >> 32) * 34001ULL) >> 32));
    return (int32_t)interp_tab(ln_dur, u); /* clipped lognormal quantile */
}

int orc_gen_trace(uint64_t seed, int32_t rate_mhz, int32_t dist, int64_t n,
                  const uint32_t *ln_dur, const uint32_t *exp_t,
                  orc_req_t *out) {
    if (rate_mhz < 1 || n < 0 || dist < 0 || dist > 1) return -1;
    /* Poisson process: exponential inter-arrival gaps */
    uint64_t mean_gap_us = 1000000000ULL / (uint64_t)rate_mhz;
    uint64_t ln2_q32 = exp_t[4096];
    int64_t t = 0;
    for (int64_t i = 0; i < n; i++) {
        uint64_t u0 = orc_mix64(seed, 0, (uint64_t)i);
        uint64_t u1 = orc_mix64(seed, 1, (uint64_t)i);
        uint64_t u2 = orc_mix64(seed, 2, (uint64_t)i);
        /* unit exponential in Q32: E = G*ln2 + E', G geometric(1/2),
         * E' exponential truncated to [0, ln 2) by inverse CDF */
        uint64_t e_q32 = (uint64_t)clz64(u0 | 1ULL) * ln2_q32 + interp_tab(exp_t, u1);
        uint64_t gap = (uint64_t)(((unsigned __int128)e_q32 * mean_gap_us) >> 32);
        t += (int64_t)gap; /* S18: first arrival = first gap after t = 0 */
        out[i].arrival_us = t;
        out[i].dur_ms = draw_duration(u2, dist, ln_dur);
        out[i].est = out[i].dur_ms; /* S7: configs set est = dur_ms */
    }
    return 0;
}

/* config-5 queues: arrival uniform in [0, now), unsorted; lognormal dur */
int orc_gen_queue(uint64_t seed, int64_t first, int64_t n, int64_t now,
                  const uint32_t *ln_dur, orc_req_t *out) {
    if (n < 0 || now < 1 || first < 0) return -1;
    for (int64_t j = 0; j < n; j++) {
        uint64_t i = (uint64_t)(first + j);
        uint64_t u2 = orc_mix64(seed, 2, i);
        uint64_t u3 = orc_mix64(seed, 3, i);
        out[j].arrival_us =
            (int64_t)(((unsigned __int128)u3 * (uint64_t)now) >> 64);
        out[j].dur_ms = draw_duration(u2, ORC_DIST_LOGNORMAL, ln_dur);
        out[j].est = out[j].dur_ms;
    }
    return 0;
}
