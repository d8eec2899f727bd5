/*
 * oracle/gemm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct fp64 CPU statement of what the hot path
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file; it shares no code, header, table or
 * helper with paper_2606_15991_b200/csrc (the CUDA path), and neither imports
 * the other.
 *
 * What it states (Listing 2 "gemm_persistent"):
 *     for every output index (bid_m, bid_n):
 *         tz = 0                                   (constant(T::ZERO))
 *         for k_tile in 0 .. num_tiles(part_x, 1):
 *             tz = mma(x[bid_m,k_tile], y[k_tile,bid_n], tz)
 *         z.store(tz, out_idx)
 * i.e. the plain definition  C_ij = sum_{k=0}^{K-1} a_ik * b_kj  with a zero
 * initial accumulator and a single store.  Edge tiles: read-only partition
 * loads are zero padded and stores are masked, so elements past
 * K contribute exactly 0 and nothing outside [0,M)x[0,N) is written.  The
 * method reaches this definition exactly up to rounding order, so the oracle
 * is the definition written out, in fp64, k ascending for every element.
 *
 * Readings taken where the paper is silent (SURVEY.md
 * section 8(c)): c1 inputs are bf16 (BASELINE.json binds; the paper measured
 * f16); c2 accumulation is wider than the element type (fp32 on the GPU, fp64
 * here); c3 y is row-major K x N; c8 K==0 gives zeros.
 *
 * Besides C the oracle returns S_ij = sum_k |a_ik|*|b_kj|, the scale of the
 * tolerance in BASELINE.json's north_star (|C_gpu - C_ref| <= 2^-5 * S).
 *
 * Why fp64 is exact enough: a bf16 x bf16 product has <= 16 significant bits
 * and is exact in fp64 (with or without FMA contraction); K <= 2^20 such terms
 * summed in fp64 carry error <= K * 2^-53 * S.  For integer-valued inputs every
 * partial sum is an exactly representable integer.
 *
 * Pins (tests/test_oracle_pins.py, all CPU): identity, all-ones (C_ij = K),
 * rank-1 closed form, k mod 8 closed form, one-hot row selection, brute force
 * on 8x8x8 against a separately written triple loop, numpy float64 matmul,
 * (AB)^T = B^T A^T, K-permutation invariance, block-size / thread-count
 * invariance, bf16 codec against torch / ml_dtypes on all 65536 patterns and
 * 10^6 random floats.  Nothing here is "parity unpinned".
 *
 * Blocking: i0 (MB rows) x k0 (KB, ascending) x j0 (NB), inner order i-k-j
 * (unit stride on B rows and C rows).  For any (i,j) the k terms are added in
 * ascending order whatever the block sizes, so block sizes and thread counts
 * cannot change a single bit.  Threads own disjoint row ranges (or, when
 * M < threads, disjoint column ranges): no cross-thread reduction.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* bf16 bit pattern -> real value.  bf16 is the upper half of an IEEE binary32. */
static inline double dec(uint16_t h)
{
    uint32_t w = ((uint32_t)h) << 16;
    float f;
    memcpy(&f, &w, sizeof f);
    return (double)f;
}

double oracle_bf16_decode(uint16_t h) { return dec(h); }

/*
 * IEEE binary16 ("f16", the precision the paper itself measures)
 * bit pattern -> real value: sign s, exponent e (5 bits, bias 15), fraction m
 * (10 bits).  e = 0: (-1)^s * m * 2^-24 (zero and subnormals); e = 31: infinity
 * (m = 0) or NaN; otherwise (-1)^s * (1 + m/1024) * 2^(e-15).
 */
static inline double dec_f16(uint16_t h)
{
    const int s = h >> 15, e = (h >> 10) & 31, m = h & 1023;
    double v;
    if (e == 0) v = (double)m * 0x1p-24;
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexp(1.0 + (double)m * 0x1p-10, e - 15);
    return s ? -v : v;
}

double oracle_f16_decode(uint16_t h) { return dec_f16(h); }

/* element type of A and B: 0 = bf16 (BASELINE.json), 1 = f16 */
static inline double dec_in(uint16_t h, const int f16) { return f16 ? dec_f16(h) : dec(h); }

/* binary32 -> bf16, round to nearest even; NaN -> quiet NaN keeping the sign. */
uint16_t oracle_bf16_encode(float f)
{
    uint32_t w;
    memcpy(&w, &f, sizeof w);
    if ((w & 0x7fffffffu) > 0x7f800000u)
        return (uint16_t)(((w >> 16) & 0x8000u) | 0x7fc0u);
    w += 0x7fffu + ((w >> 16) & 1u);
    return (uint16_t)(w >> 16);
}

void oracle_bf16_decode_array(const uint16_t *src, double *dst, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) dst[i] = dec(src[i]);
}

void oracle_bf16_encode_array(const float *src, uint16_t *dst, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) dst[i] = oracle_bf16_encode(src[i]);
}

void oracle_f16_decode_array(const uint16_t *src, double *dst, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) dst[i] = dec_f16(src[i]);
}

typedef struct {
    const uint16_t *A, *B;
    double *C, *S;
    int64_t i_lo, i_hi, j_lo, j_hi, K, lda, ldb, ldc;
    int64_t MB, KB, NB;
    int f16; /* input element type, see dec_in */
} range_job;

static inline int64_t min64(int64_t a, int64_t b) { return a < b ? a : b; }

/* One thread's share: rows [i_lo,i_hi) x columns [j_lo,j_hi), all of K.  `f16` is a
 * compile-time constant in both callers, so the decode is resolved outside the loops. */
static inline void run_range_typed(const range_job *q, const int f16)
{
    for (int64_t i = q->i_lo; i < q->i_hi; ++i)
        for (int64_t j = q->j_lo; j < q->j_hi; ++j) {
            q->C[i * q->ldc + j] = 0.0; /* tz = constant(ZERO) */
            q->S[i * q->ldc + j] = 0.0;
        }
    for (int64_t i0 = q->i_lo; i0 < q->i_hi; i0 += q->MB)
        for (int64_t k0 = 0; k0 < q->K; k0 += q->KB)
            for (int64_t j0 = q->j_lo; j0 < q->j_hi; j0 += q->NB) {
                const int64_t i1 = min64(i0 + q->MB, q->i_hi);
                const int64_t k1 = min64(k0 + q->KB, q->K);
                const int64_t j1 = min64(j0 + q->NB, q->j_hi);
                for (int64_t i = i0; i < i1; ++i) {
                    double *c = q->C + i * q->ldc;
                    double *s = q->S + i * q->ldc;
                    for (int64_t k = k0; k < k1; ++k) {
                        const double a = dec_in(q->A[i * q->lda + k], f16);
                        const double aa = fabs(a);
                        const uint16_t *b = q->B + k * q->ldb;
                        for (int64_t j = j0; j < j1; ++j) {
                            const double bv = dec_in(b[j], f16);
                            c[j] += a * bv;        /* tz = mma(tx, ty, tz) */
                            s[j] += aa * fabs(bv); /* tolerance scale      */
                        }
                    }
                }
            }
}

static void *run_range(void *arg)
{
    const range_job *q = (const range_job *)arg;
    if (q->f16) run_range_typed(q, 1);
    else run_range_typed(q, 0);
    return NULL;
}

/*
 * Full problem.  A: M x K bf16 bit patterns, row stride lda; B: K x N, row
 * stride ldb; C,S: M x N fp64, row stride ldc (all strides in elements).
 * threads <= 0 means 1.  MB/KB/NB <= 0 select 64/256/512.  Returns 0, or -1 on
 * a bad argument.
 */
int oracle_gemm_typed(const uint16_t *A, const uint16_t *B, double *C, double *S,
                      int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
                      int64_t ldc, int threads, int64_t MB, int64_t KB, int64_t NB,
                      int in_f16)
{
    if (M < 0 || N < 0 || K < 0 || lda < K || ldb < N || ldc < N) return -1;
    if (M == 0 || N == 0) return 0;
    if (threads <= 0) threads = 1;
    if (threads > 256) threads = 256;
    if (MB <= 0) MB = 64;
    if (KB <= 0) KB = 256;
    if (NB <= 0) NB = 512;

    range_job jobs[256];
    pthread_t tid[256];
    int n = 0;
    if (M >= threads) { /* disjoint row ranges */
        const int64_t per = (M + threads - 1) / threads;
        for (int t = 0; t < threads; ++t) {
            const int64_t lo = t * per, hi = min64(lo + per, M);
            if (lo >= hi) break;
            jobs[n++] = (range_job){A, B, C, S, lo, hi, 0, N, K, lda, ldb, ldc, MB, KB, NB, in_f16 != 0};
        }
    } else { /* few rows (the M=1 GEMV): disjoint column ranges */
        const int64_t per = (N + threads - 1) / threads;
        for (int t = 0; t < threads; ++t) {
            const int64_t lo = t * per, hi = min64(lo + per, N);
            if (lo >= hi) break;
            jobs[n++] = (range_job){A, B, C, S, 0, M, lo, hi, K, lda, ldb, ldc, MB, KB, NB, in_f16 != 0};
        }
    }
    if (n == 1) {
        run_range(&jobs[0]);
        return 0;
    }
    for (int t = 0; t < n; ++t)
        if (pthread_create(&tid[t], NULL, run_range, &jobs[t]) != 0) {
            for (int u = 0; u < t; ++u) pthread_join(tid[u], NULL);
            return -1;
        }
    for (int t = 0; t < n; ++t) pthread_join(tid[t], NULL);
    return 0;
}

/* bf16 inputs (BASELINE.json's five configs). */
int oracle_gemm(const uint16_t *A, const uint16_t *B, double *C, double *S,
                int64_t M, int64_t N, int64_t K, int64_t lda, int64_t ldb,
                int64_t ldc, int threads, int64_t MB, int64_t KB, int64_t NB)
{
    return oracle_gemm_typed(A, B, C, S, M, N, K, lda, ldb, ldc, threads, MB, KB, NB, 0);
}

/*
 * Sampled variant: for each listed (i,j) the two dot products over
 * k = 0..K-1, k ascending, directly from the definition.
 */
int oracle_gemm_sampled_typed(const uint16_t *A, const uint16_t *B, const int64_t *si,
                              const int64_t *sj, int64_t nsamples, double *c_out,
                              double *s_out, int64_t M, int64_t N, int64_t K,
                              int64_t lda, int64_t ldb, int in_f16)
{
    if (M < 0 || N < 0 || K < 0 || lda < K || ldb < N) return -1;
    for (int64_t t = 0; t < nsamples; ++t) {
        const int64_t i = si[t], j = sj[t];
        if (i < 0 || i >= M || j < 0 || j >= N) return -1;
        double c = 0.0, s = 0.0;
        for (int64_t k = 0; k < K; ++k) {
            const double a = dec_in(A[i * lda + k], in_f16 != 0);
            const double b = dec_in(B[k * ldb + j], in_f16 != 0);
            c += a * b;
            s += fabs(a) * fabs(b);
        }
        c_out[t] = c;
        s_out[t] = s;
    }
    return 0;
}

int oracle_gemm_sampled(const uint16_t *A, const uint16_t *B, const int64_t *si,
                        const int64_t *sj, int64_t nsamples, double *c_out,
                        double *s_out, int64_t M, int64_t N, int64_t K,
                        int64_t lda, int64_t ldb)
{
    return oracle_gemm_sampled_typed(A, B, si, sj, nsamples, c_out, s_out, M, N, K, lda, ldb, 0);
}
