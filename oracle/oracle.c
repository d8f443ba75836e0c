/*
 * oracle.c -- fp64 CPU oracle for MaxSim scoring.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain definition of what the CUDA path must compute, written out from the
 * paper (/root/reference/PAPER.md, cited as P:L<line>).  It shares no code, headers, tables or
 * helpers with paper_2606_26439_b200/csrc and must never be linked into or called from the
 * product path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.
 *
 * What it computes
 *   dense  (Eq. 1):   score(q,b) = sum_{i<Nq}  max_{j in doc b}  q_i^T d_j
 *   PQ     ("decompress, then score"; Eq. 8-9 P:L255-262 define the same value):
 *          d^_t = concat_m C[m, codes[t,m], :]   then the dense definition on d^.
 *
 * Precision: inputs are the storage-dtype bytes the GPU sees (fp32 / fp16 / bf16), converted
 * EXACTLY to fp64; every multiply, add and compare is fp64; the dot product runs k ascending,
 * the sum over query tokens i ascending.  Compiled with -ffp-contract=off so no FMA contraction
 * changes the rounding between the two implementations below.
 *
 * Readings of the paper taken here: raw dot product, no normalisation
 * (A1); an empty document scores -inf, the literal outcome of m <- -inf (Alg. 3 line 4)
 * (A2); every one of the Nq query rows counts (A5).
 *
 * Pins (tests/test_oracle_pins.py): brute force vs the transposed form (bit-identical), numpy
 * float64 einsum on tiny inputs, self-retrieval = sum ||q_i||^2, permutation invariance,
 * |score| <= Nq for unit norm, one-hot queries = sum of column maxima, single-token documents =
 * GEMV, additivity over query tokens, zero-padded d, homogeneity, PQ LUT identity (Eq. 9),
 * lossless PQ = dense.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* dtype codes: the numeric values of the public enum are part of the C-ABI contract, restated here */
enum { ORACLE_F32 = 0, ORACLE_F16 = 1, ORACLE_BF16 = 2 };

/* ---- exact element decoding, written here independently of the CUDA path ---------------------- */

/* bfloat16: the upper 16 bits of an IEEE binary32 */
static double decode_bf16(uint16_t h) {
    uint32_t w = ((uint32_t)h) << 16;
    float f;
    memcpy(&f, &w, sizeof f);
    return (double)f;
}

/* IEEE binary16: 1 sign, 5 exponent (bias 15), 10 mantissa bits; subnormals and +-0 handled */
static double decode_f16(uint16_t h) {
    int sign = (h >> 15) & 1;
    int expo = (h >> 10) & 0x1f;
    int mant = h & 0x3ff;
    double v;
    if (expo == 0) {
        v = ldexp((double)mant, -24); /* subnormal: mant * 2^-10 * 2^-14 */
    } else if (expo == 31) {
        v = mant ? NAN : INFINITY; /* outside the contract (A8) but decoded faithfully */
    } else {
        v = ldexp(1.0 + (double)mant / 1024.0, expo - 15);
    }
    return sign ? -v : v;
}

static double decode_elem(const void* base, int64_t idx, int dtype) {
    switch (dtype) {
        case ORACLE_F32: return (double)((const float*)base)[idx];
        case ORACLE_F16: return decode_f16(((const uint16_t*)base)[idx]);
        default: return decode_bf16(((const uint16_t*)base)[idx]);
    }
}

static size_t elem_size(int dtype) { return dtype == ORACLE_F32 ? 4 : 2; }

/* ---- P1: the literal nested loops of Eq. 1, one thread, no scratch -------------------- */

void oracle_bruteforce(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets,
                       int64_t B, int dtype, double* scores) {
    for (int q = 0; q < Q; ++q) {
        for (int64_t b = 0; b < B; ++b) {
            double total = 0.0;
            for (int i = 0; i < Nq; ++i) {
                double m = -INFINITY; /* Alg. 3 line 4: m <- -inf */
                for (int64_t t = offsets[b]; t < offsets[b + 1]; ++t) {
                    double s = 0.0;
                    for (int k = 0; k < d; ++k) {
                        double a = decode_elem(queries, ((int64_t)q * Nq + i) * d + k, dtype);
                        double c = decode_elem(docs, t * d + k, dtype);
                        s = s + a * c;
                    }
                    if (s > m) m = s;
                }
                total = total + m;
            }
            scores[(int64_t)q * B + b] = total;
        }
    }
}

/* ---- the same definition, document decoded once and transposed so the j loop is innermost ------ */
/* Every s_ij still accumulates k = 0..d-1 in order, so the result is bit-identical to the brute   */
/* force; only the loop nest is interchanged (k outer, j inner) and documents run in parallel.     */

static void score_one_doc(const double* qd /* [Q*Nq, d] */, int Q, int Nq, int d, const double* Dt /* [d, nd] */,
                          int64_t nd, double* s /* [nd] scratch */, double* out /* stride B */, int64_t B) {
    for (int q = 0; q < Q; ++q) {
        double total = 0.0;
        for (int i = 0; i < Nq; ++i) {
            const double* qi = qd + ((int64_t)q * Nq + i) * d;
            for (int64_t j = 0; j < nd; ++j) s[j] = 0.0;
            for (int k = 0; k < d; ++k) {
                const double a = qi[k];
                const double* row = Dt + (int64_t)k * nd;
                for (int64_t j = 0; j < nd; ++j) s[j] = s[j] + a * row[j];
            }
            double m = -INFINITY;
            for (int64_t j = 0; j < nd; ++j)
                if (s[j] > m) m = s[j];
            total = total + m;
        }
        out[(int64_t)q * B] = total;
    }
}

static int64_t max_doc_len(const int64_t* offsets, int64_t B) {
    int64_t mx = 0;
    for (int64_t b = 0; b < B; ++b) {
        int64_t n = offsets[b + 1] - offsets[b];
        if (n > mx) mx = n;
    }
    return mx;
}

/* returns the number of threads actually used */
int oracle_maxsim(const void* queries, int Q, int Nq, int d, const void* docs, const int64_t* offsets, int64_t B,
                  int dtype, double* scores, int threads) {
    const int64_t nrows = (int64_t)Q * Nq;
    double* qd = (double*)malloc(sizeof(double) * (size_t)(nrows * d > 0 ? nrows * d : 1));
    for (int64_t e = 0; e < nrows * d; ++e) qd[e] = decode_elem(queries, e, dtype);
    const int64_t mx = max_doc_len(offsets, B);
    int used = 1;
    (void)threads;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#pragma omp parallel
#endif
    {
#ifdef _OPENMP
#pragma omp single
        used = omp_get_num_threads();
#endif
        double* Dt = (double*)malloc(sizeof(double) * (size_t)(mx * d > 0 ? mx * d : 1));
        double* s = (double*)malloc(sizeof(double) * (size_t)(mx > 0 ? mx : 1));
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 16)
#endif
        for (int64_t b = 0; b < B; ++b) {
            const int64_t t0 = offsets[b], nd = offsets[b + 1] - offsets[b];
            for (int64_t j = 0; j < nd; ++j)
                for (int k = 0; k < d; ++k) Dt[(int64_t)k * nd + j] = decode_elem(docs, (t0 + j) * d + k, dtype);
            score_one_doc(qd, Q, Nq, d, Dt, nd, s, scores + b, B);
        }
        free(Dt);
        free(s);
    }
    free(qd);
    return used;
}

/* ---- PQ: explicit decompression, then the dense definition --------------------------- */
/* No lookup table is built here; Eq. 9's identity is checked against this by a separate fp64      */
/* table in the tests (pin P5).                                                                    */

int oracle_pq_maxsim(const void* queries, int Q, int Nq, int d, int q_dtype, const float* codebooks /* [M,K,d/M] */,
                     int M, int K, const uint8_t* codes /* [T, M] */, const int64_t* offsets, int64_t B,
                     double* scores, int threads) {
    const int dsub = d / M;
    const int64_t nrows = (int64_t)Q * Nq;
    double* qd = (double*)malloc(sizeof(double) * (size_t)(nrows * d > 0 ? nrows * d : 1));
    for (int64_t e = 0; e < nrows * d; ++e) qd[e] = decode_elem(queries, e, q_dtype);
    const int64_t mx = max_doc_len(offsets, B);
    int used = 1;
    (void)threads;
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#pragma omp parallel
#endif
    {
#ifdef _OPENMP
#pragma omp single
        used = omp_get_num_threads();
#endif
        float* dhat = (float*)malloc(sizeof(float) * (size_t)(mx * d > 0 ? mx * d : 1)); /* the decompressed doc */
        double* Dt = (double*)malloc(sizeof(double) * (size_t)(mx * d > 0 ? mx * d : 1));
        double* s = (double*)malloc(sizeof(double) * (size_t)(mx > 0 ? mx : 1));
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 16)
#endif
        for (int64_t b = 0; b < B; ++b) {
            const int64_t t0 = offsets[b], nd = offsets[b + 1] - offsets[b];
            /* step 1: d^_t = concat_m C[m, codes[t,m], 0:dsub], an exact fp32 copy */
            for (int64_t j = 0; j < nd; ++j)
                for (int m = 0; m < M; ++m) {
                    const int c = codes[(t0 + j) * M + m];
                    (void)K;
                    memcpy(dhat + j * d + (int64_t)m * dsub, codebooks + ((int64_t)m * K + c) * dsub,
                           sizeof(float) * (size_t)dsub);
                }
            /* step 2: the dense definition on d^ */
            for (int64_t j = 0; j < nd; ++j)
                for (int k = 0; k < d; ++k) Dt[(int64_t)k * nd + j] = (double)dhat[j * d + k];
            score_one_doc(qd, Q, Nq, d, Dt, nd, s, scores + b, B);
        }
        free(dhat);
        free(Dt);
        free(s);
    }
    free(qd);
    return used;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
