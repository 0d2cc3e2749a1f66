/*
 * dpi_oracle.c -- plain, slow, obviously-correct CPU oracle for the fused multi-table embedding lookup
 * of DPIFrame (arxiv 2606.21101).  TEST INFRASTRUCTURE ONLY: nothing on the product path may call it;
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs do.
 * It shares no code, header, table or helper with paper_2606_21101_b200/csrc/ and neither imports the other.
 *
 * What it follows (line numbers are /root/reference/PAPER.md):
 *   - Algorithm 1 "Multi-table Lookup" (prose 139-141 and 166): for every element idx of
 *     EmbedOut[b x (k*d)]: row = idx / (k*d); col = idx mod (k*d); table_id = col / d;
 *     emb_row = IDs[row*k + table_id]; emb_col = col mod d;
 *     EmbedOut[idx] = Embs[table_id][emb_row*d + emb_col].            -> oracle_alg1_onehot()
 *   - Multi-hot "by marking offset information" read as CSR bags with sum / mean pooling
 *     (readings R2, R7, R8): out[b, t*D + c] = sum_{j in bag(b,t)} E_t[indices[j]][c],
 *     divided by the bag length for mean tables, all-zero for an empty bag.   -> oracle_lookup()
 *   - "The overall embedding workload is deterministic and known in advance": the whole
 *     workload is laid out before the pass.  North-star planner = exclusive scan of bag lengths plus
 *     balanced contiguous segments of cost ~K (DESIGN.md §3 gives the closed integer definition).
 *                                                                              -> oracle_plan()
 * Arithmetic: float64 accumulation, result kept UNROUNDED (double).  Loop order t -> b -> j -> c exactly as
 * written in DESIGN.md §4; no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Alg. 1 gather identity and column-block order via
 * index-encoding tables, the hand-worked Fig.-5-shaped fixture tests/golden/fig5_shape_example.txt,
 * constant / row-id tables (closed forms), mean == sum/len, empty bag == +0.0, the one-hot-matrix product
 * formulation ("encoded with one-hot encoding") via numpy matmul, torch-CPU embedding_bag,
 * table independence, sample permutation, numpy cumsum, closed form for equal lengths,
 * cover/monotone/bounded-cost invariants, O(G*S) brute force, and exhaustive 16-bit decode checks.
 * oracle_lookup_general (interface variants) is pinned in tests/test_oracle_variants.py: torch-CPU embedding_bag
 * with per_sample_weights (float64), linearity / power-of-two / zero weights, index-encoding tables with mixed
 * dims, hstack of single-table calls, and the bag-grid transpose for table-major input.
 * oracle_plan_stats (min / max bag length, a1's "uniform-length flag") and oracle_plan64 (64-bit offsets, N >= 2^31) are
 * pinned in tests/test_oracle_plan.py: the hand-worked fixture, closed forms for constant and arithmetic-progression
 * lengths (incl. lengths whose sum passes 2^31), permutation / concatenation invariants, sorted-order brute force and
 * equality with the 32-bit plan wherever both are defined.
 * oracle_lookup_par is oracle_lookup with the two outer loops interchanged (samples outside, OpenMP over samples); every
 * bag is pooled by the same pool_bag() in the same j -> c order, so the block is bit-identical -- pinned by exactly that
 * equality in tests/test_oracle_lookup.py. It exists only so that bench.py can time the oracle on all host cores.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

enum { ORACLE_F32 = 0, ORACLE_F16 = 1, ORACLE_BF16 = 2 };
enum { ORACLE_SUM = 0, ORACLE_MEAN = 1 };
enum { ORACLE_OK = 0, ORACLE_BAD_ARG = 1, ORACLE_INDEX_RANGE = 2, ORACLE_OVERFLOW = 3, ORACLE_CAPACITY = 4 };

/* IEEE binary16 -> double, by hand (sign | 5-bit exponent | 10-bit fraction). */
static double half_bits_to_double(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int e = (h >> 10) & 0x1F;
    int f = h & 0x3FF;
    double v;
    if (e == 0) {
        v = (double)f * (1.0 / 16777216.0);               /* subnormal: f * 2^-24 */
    } else if (e == 31) {
        v = f ? (0.0 / 0.0) : (1.0 / 0.0);                /* NaN / Inf (never produced by the generators) */
    } else {
        double m = 1.0 + (double)f * (1.0 / 1024.0);
        double s = 1.0;
        int k = e - 15;
        while (k > 0) { s *= 2.0; --k; }
        while (k < 0) { s *= 0.5; ++k; }
        v = m * s;
    }
    return sign ? -v : v;
}

/* bfloat16 = upper 16 bits of an IEEE binary32. */
static double bf16_bits_to_double(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

static double element_as_double(const void *table, int dtype, int64_t pos)
{
    switch (dtype) {
    case ORACLE_F32:  return (double)((const float *)table)[pos];
    case ORACLE_F16:  return half_bits_to_double(((const uint16_t *)table)[pos]);
    default:          return bf16_bits_to_double(((const uint16_t *)table)[pos]);
    }
}

/* exported for the exhaustive decoder pins */
double oracle_decode_f16(uint16_t h)  { return half_bits_to_double(h); }
double oracle_decode_bf16(uint16_t b) { return bf16_bits_to_double(b); }

/*
 * Algorithm 1, literally: one-hot IDs[b x k], per-table local ids, common d.
 * Lines 4-6 are garbled in the extracted text; reconstructed from the prose at PAPER.md:141 and 166
 * (reading R1).
 */
int oracle_alg1_onehot(int32_t b, int32_t k, int32_t d, int dtype,
                       const void *const *Embs, const int64_t *n_rows,
                       const int32_t *IDs, double *EmbedOut)
{
    if (b < 0 || k <= 0 || d <= 0 || !Embs || !IDs || !EmbedOut) return ORACLE_BAD_ARG;
    int64_t total_elements = (int64_t)b * k * d;                 /* line 1 */
    int64_t row_width = (int64_t)k * d;                          /* line 2 */
    for (int64_t idx = 0; idx < total_elements; ++idx) {         /* line 3 */
        int64_t row = idx / row_width;                           /* line 4 */
        int64_t col = idx % row_width;                           /* line 5 */
        int64_t table_id = col / d;                              /* line 6 */
        int64_t emb_row = IDs[row * k + table_id];               /* line 7 */
        int64_t emb_col = col % d;                               /* line 8 */
        if (emb_row < 0 || (n_rows && emb_row >= n_rows[table_id])) return ORACLE_INDEX_RANGE;
        EmbedOut[idx] = element_as_double(Embs[table_id], dtype, emb_row * d + emb_col);   /* line 9 */
    }
    return ORACLE_OK;                                            /* line 11 */
}

/*
 * Pooled multi-hot lookup.  Bag g = b*T + t owns indices[offsets[g] .. offsets[g+1]).
 * ref is [B, T*D] row-major float64, table t at columns [t*D, (t+1)*D).
 */
/* One bag (b, t): the inner two loops of DESIGN.md §4 (entries j in order, columns c), float64, unrounded. */
static int pool_bag(int32_t T, int32_t D, int dtype, const void *table, int64_t rows_t, int pool_t,
                    const int32_t *indices, const int32_t *offsets, int32_t b, int32_t t, double *ref)
{
    int64_t g = (int64_t)b * T + t;
    int64_t lo = offsets[g], hi = offsets[g + 1];
    double *acc = ref + (int64_t)b * ((int64_t)T * D) + (int64_t)t * D;
    if (hi < lo) return ORACLE_BAD_ARG;
    for (int32_t c = 0; c < D; ++c) acc[c] = 0.0;
    for (int64_t j = lo; j < hi; ++j) {
        int64_t r = indices[j];
        if (r < 0 || r >= rows_t) return ORACLE_INDEX_RANGE;
        for (int32_t c = 0; c < D; ++c)
            acc[c] += element_as_double(table, dtype, r * D + c);
    }
    if (pool_t == ORACLE_MEAN && hi > lo) {
        double L = (double)(hi - lo);
        for (int32_t c = 0; c < D; ++c) acc[c] /= L;
    }
    return ORACLE_OK;
}

int oracle_lookup(int32_t T, int32_t B, int32_t D, int dtype,
                  const void *const *tables, const int64_t *table_rows,
                  const int32_t *indices, const int32_t *offsets,
                  const uint8_t *pooling, double *ref)
{
    if (T <= 0 || B < 0 || D <= 0 || !tables || !table_rows || !offsets || !pooling || !ref) return ORACLE_BAD_ARG;
    if (dtype != ORACLE_F32 && dtype != ORACLE_F16 && dtype != ORACLE_BF16) return ORACLE_BAD_ARG;
    for (int32_t t = 0; t < T; ++t) {                            /* tables in order -> column block t */
        for (int32_t b = 0; b < B; ++b) {                        /* samples -> output row b */
            int rc = pool_bag(T, D, dtype, tables[t], table_rows[t], pooling[t], indices, offsets, b, t, ref);
            if (rc != ORACLE_OK) return rc;
        }
    }
    return ORACLE_OK;
}

/*
 * The same lookup on all host cores, for bench.py's cpu_baseline only (SURVEY.md 8(d) "Oracle timing" (ii)): bags are
 * independent, so the sample loop is moved outside and split over threads; each bag still goes through
 * pool_bag() in the same entry and column order, hence the block is bit-identical to oracle_lookup's.
 * threads_used receives the team size (may be NULL). Compiled without OpenMP this is a plain loop.
 */
#ifdef _OPENMP
#include <omp.h>
#endif
int oracle_lookup_par(int32_t T, int32_t B, int32_t D, int dtype,
                      const void *const *tables, const int64_t *table_rows,
                      const int32_t *indices, const int32_t *offsets,
                      const uint8_t *pooling, double *ref, int32_t *threads_used)
{
    if (T <= 0 || B < 0 || D <= 0 || !tables || !table_rows || !offsets || !pooling || !ref) return ORACLE_BAD_ARG;
    if (dtype != ORACLE_F32 && dtype != ORACLE_F16 && dtype != ORACLE_BF16) return ORACLE_BAD_ARG;
    int status = ORACLE_OK;
    int team = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        team = omp_get_num_threads();
#pragma omp for schedule(static)
#endif
        for (int32_t b = 0; b < B; ++b) {
            for (int32_t t = 0; t < T; ++t) {
                int rc = pool_bag(T, D, dtype, tables[t], table_rows[t], pooling[t], indices, offsets, b, t, ref);
                if (rc != ORACLE_OK) {
#ifdef _OPENMP
#pragma omp critical
#endif
                    status = rc;
                }
            }
        }
#ifdef _OPENMP
    }
#endif
    if (threads_used) *threads_used = team;
    return status;
}

/*
 * Interface variants of the same lookup (DESIGN.md §11 gives the readings).  The paper
 * only hints at them: multi-hot "by marking offset information" and ids arriving as 64-bit
 * integers from the framework.  Same definition as oracle_lookup with four generalisations:
 *   dims[t]      per-table embedding dim; table t occupies columns [col[t], col[t] + dims[t]) of a row of width
 *                W = sum dims, col[t] = sum_{u<t} dims[u]            ("concatenated", one d at :137)
 *   bag_order    0: sample-major, bag (b,t) is g = b*T + t  (Alg. 1 line 7)
 *                1: table-major,  bag (b,t) is g = t*B + b  (all bags of field 0, then field 1, ...)
 *   indices / offsets are int64
 *   weights      NULL, or one fp32 weight per index entry: acc += w[j] * E_t[indices[j]]  (sum pooling only;
 *                a mean-pooled table together with weights is rejected)
 * ref is [B, W] row-major float64, unrounded.  Loop order t -> b -> j -> c as in oracle_lookup.
 */
int oracle_lookup_general(int32_t T, int32_t B, const int32_t *dims, int dtype,
                          const void *const *tables, const int64_t *table_rows,
                          const int64_t *indices, const int64_t *offsets, const float *weights,
                          const uint8_t *pooling, int bag_order, double *ref)
{
    if (T <= 0 || B < 0 || !dims || !tables || !table_rows || !offsets || !pooling || !ref) return ORACLE_BAD_ARG;
    if (dtype != ORACLE_F32 && dtype != ORACLE_F16 && dtype != ORACLE_BF16) return ORACLE_BAD_ARG;
    if (bag_order != 0 && bag_order != 1) return ORACLE_BAD_ARG;
    int64_t W = 0;
    for (int32_t t = 0; t < T; ++t) {
        if (dims[t] <= 0) return ORACLE_BAD_ARG;
        if (weights && pooling[t] == ORACLE_MEAN) return ORACLE_BAD_ARG;
        W += dims[t];
    }
    int64_t col = 0;                                             /* col[t] */
    for (int32_t t = 0; t < T; ++t) {
        int32_t D = dims[t];
        for (int32_t b = 0; b < B; ++b) {
            int64_t g = bag_order == 0 ? (int64_t)b * T + t : (int64_t)t * B + b;
            int64_t lo = offsets[g], hi = offsets[g + 1];
            double *acc = ref + (int64_t)b * W + col;
            if (hi < lo) return ORACLE_BAD_ARG;
            for (int32_t c = 0; c < D; ++c) acc[c] = 0.0;
            for (int64_t j = lo; j < hi; ++j) {
                int64_t r = indices[j];
                double w = weights ? (double)weights[j] : 1.0;
                if (r < 0 || r >= table_rows[t]) return ORACLE_INDEX_RANGE;
                for (int32_t c = 0; c < D; ++c)
                    acc[c] += w * element_as_double(tables[t], dtype, r * D + c);
            }
            if (pooling[t] == ORACLE_MEAN && hi > lo) {
                double L = (double)(hi - lo);
                for (int32_t c = 0; c < D; ++c) acc[c] /= L;
            }
        }
        col += D;
    }
    return ORACLE_OK;
}

/*
 * Workload plan:
 *   offsets[0] = 0; offsets[g+1] = offsets[g] + len[g]                 (int32; N < 2^31 required)
 *   C[0] = 0;       C[g+1] = C[g] + max(len[g], 1)                     (an empty bag still costs one store)
 *   S = ceil(C[G] / K)
 *   seg_bag[s] = min(G, min{ g in [0,G] : C[g] >= s*K }),  s = 0..S
 *   seg_off[s] = offsets[seg_bag[s]]                        (first index entry of task s; may be NULL)
 * seg_cap is the capacity of seg_bag / seg_off in elements (needs S+1).
 */
int oracle_plan(const int32_t *len, int64_t G, int32_t K,
                int32_t *offsets, int32_t *seg_bag, int32_t *seg_off, int64_t seg_cap, int32_t *S_out)
{
    if (!len || G < 0 || K < 1 || !offsets || !seg_bag || !S_out) return ORACLE_BAD_ARG;
    int64_t off = 0;
    offsets[0] = 0;
    for (int64_t g = 0; g < G; ++g) {
        if (len[g] < 0) return ORACLE_BAD_ARG;
        off += len[g];
        if (off > 2147483647LL) return ORACLE_OVERFLOW;
        offsets[g + 1] = (int32_t)off;
    }
    /* total cost C[G] */
    int64_t CG = 0;
    for (int64_t g = 0; g < G; ++g) CG += (len[g] > 1 ? len[g] : 1);
    int64_t S = (CG + K - 1) / K;
    if (S + 1 > seg_cap) return ORACLE_CAPACITY;
    /* seg_bag[s]: smallest g with C[g] >= s*K; the target s*K grows with s, so g only moves forward */
    int64_t g = 0, Cg = 0;                                       /* Cg == C[g] */
    for (int64_t s = 0; s <= S; ++s) {
        int64_t target = s * (int64_t)K;
        while (g < G && Cg < target) {
            Cg += (len[g] > 1 ? len[g] : 1);
            ++g;
        }
        /* here either Cg >= target (g is the lower bound) or g == G with C[G] < target (clamped to G) */
        seg_bag[s] = (int32_t)g;
        if (seg_off) seg_off[s] = offsets[g];
    }
    *S_out = (int32_t)S;
    return ORACLE_OK;
}

/*
 * a1's summary of the length sequence (SURVEY.md 8(a) a1 "min/max len (uniform-length flag)"; "the overall embedding
 * workload is deterministic and known in advance", PAPER.md:109 -- the one-hot workload of Alg. 1 is the case
 * min_len == max_len == 1).  DESIGN.md §3:
 *   min_len = min_{g in [0,G)} len[g],  max_len = max_{g in [0,G)} len[g];   G == 0 -> both 0.
 */
int oracle_plan_stats(const int32_t *len, int64_t G, int32_t *min_len, int32_t *max_len)
{
    if ((!len && G > 0) || G < 0 || !min_len || !max_len) return ORACLE_BAD_ARG;
    int32_t lo = 0, hi = 0;
    for (int64_t g = 0; g < G; ++g) {
        if (len[g] < 0) return ORACLE_BAD_ARG;
        if (g == 0 || len[g] < lo) lo = len[g];
        if (g == 0 || len[g] > hi) hi = len[g];
    }
    *min_len = lo;
    *max_len = hi;
    return ORACLE_OK;
}

/*
 * The same plan with 64-bit offsets (SURVEY.md 8(f) NEXT-2 "int64 indices/offsets"; ids and offsets reach the model as
 * 64-bit integers): identical definition to oracle_plan, only offsets[], seg_off[] and S are
 * int64, so N = sum len may be >= 2^31.  G < 2^31 still (seg_bag stays int32).
 */
int oracle_plan64(const int32_t *len, int64_t G, int64_t K,
                  int64_t *offsets, int32_t *seg_bag, int64_t *seg_off, int64_t seg_cap, int64_t *S_out)
{
    if (!len || G < 0 || G > 2147483647LL || K < 1 || !offsets || !seg_bag || !S_out) return ORACLE_BAD_ARG;
    offsets[0] = 0;
    for (int64_t g = 0; g < G; ++g) {
        if (len[g] < 0) return ORACLE_BAD_ARG;
        offsets[g + 1] = offsets[g] + len[g];
    }
    int64_t CG = 0;
    for (int64_t g = 0; g < G; ++g) CG += (len[g] > 1 ? len[g] : 1);
    int64_t S = (CG + K - 1) / K;
    if (S + 1 > seg_cap) return ORACLE_CAPACITY;
    int64_t g = 0, Cg = 0;
    for (int64_t s = 0; s <= S; ++s) {
        int64_t target = s * K;
        while (g < G && Cg < target) {
            Cg += (len[g] > 1 ? len[g] : 1);
            ++g;
        }
        seg_bag[s] = (int32_t)g;
        if (seg_off) seg_off[s] = offsets[g];
    }
    *S_out = S;
    return ORACLE_OK;
}
