/*
 * twq_oracle.c -- CPU ORACLE for the TwinQuant dual-component linear layer.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under paper_2606_01556_b200/ may include,
 * link, import or call this file; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs use it.  It shares no code,
 * header, table or helper with the CUDA path.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, arxiv 2606.01556):
 *   Y = deq(Q4(X*T) * R4^T) + (X*L1)*L2
 * i.e. the inference form of Eq. 3 (section 2) with the 4-bit
 * symmetric group quantizer of Eq. 1 (L43-47), the quantized product of Eq. 2
 * (L49-50), group size G along the reduction axis (L193, section 5.1), INT32-
 * style exact integer accumulation (L177) and one final merge of the two
 * components (L181, section 4.3).  The low-rank branch is the two-stage
 * high-precision product BASELINE.json's north_star fixes (SVDQuant form,
 * PAPER.md L177 "keeps the low-rank path in FP16"); it reads the raw X.
 *
 * Plain, slow, step by step in the paper's order.  No blocking, no fusion, no
 * reordering.  Floating point: the quantizer is FP32 in the exact op sequence
 * listed in DESIGN.md "Readings" R8 (that sequence is part of the spec, the
 * CUDA path must reproduce its bits); everything downstream is exact int64 or
 * FP64.  Build: gcc -O2 -fopenmp -ffp-contract=off (NO -ffast-math).
 *
 * Parity pins (tests/test_oracle_pins.py): Eq. 1 closed form and round-trip
 * bound, sign / power-of-two scaling invariances, nibble bijection, brute
 * force with python Fractions, numpy int64 matmul for P, numpy FP64 matmul for
 * the low-rank branch, r=0 and R=0 special cases, additivity, storage ratios
 * of PAPER.md L86; twq_oracle_forward_q4lr (NEXT-1, the paper's 4-bit low-rank branch): library
 * integer matmul + explicit fold for H, numpy FP32 restatement of the re-quantizer, exact closed form,
 * zero-factor reduction, round-trip bound.  The paper prints no worked numerical example, so the
 * readings R5 (rounding mode), R8 (op order), R9 (zero group), R10 (nibble
 * order) are "parity unpinned" BY THE PAPER and fixed by DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- storage formats -> arithmetic types (exact conversions) ------------- */
static float bf16_to_f32(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

static double fp16_to_f64(uint16_t h) {
    int sign = (h >> 15) & 1;
    int e = (h >> 10) & 0x1F;
    int m = h & 0x3FF;
    double v;
    if (e == 0)       v = ldexp((double)m, -24);              /* subnormal / zero */
    else if (e == 31) v = m ? NAN : INFINITY;
    else              v = ldexp((double)(m + 1024), e - 25);
    return sign ? -v : v;
}

/* ---- step 1-3: activation-side transform + group quantizer ---------------
 * PAPER.md L43-47 Eq. 1:  Q_X = round(X / s_X),  s_X = max|X| / q_max,
 * q_max = 2^(k-1)-1 = 7 for k = 4;  per-channel scaling X*diag(lambda)^-1 is
 * the activation-side transform (L54-58); groups of G contiguous elements
 * along K share one scale (L193).
 *   x~   = (float)X[m,k]            (BF16 -> FP32, exact)
 *   x~   = x~ * tinv[k]             (one FP32 RN multiply; skipped if tinv==NULL)
 *   amax = max_k |x~|  over the group (exact)
 *   amax = max(amax, 2^-30)         (R9: zero group -> codes 0, no div by 0)
 *   s    = amax / 7.0f              (FP32 RN divide)  -> sx[m,g]
 *   inv  = 1.0f / s                 (FP32 RN divide)
 *   q    = clamp((int)nearbyintf(x~ * inv), -7, 7)   (FP32 RN multiply, RNE)
 * q is int8 [M,K]; sx is float [M,K/G].
 */
void twq_oracle_quantize_act(const uint16_t* X, int M, int K, int ldx,
                             const float* tinv, int G, int8_t* q, float* sx) {
    int ng = K / G;
    for (int m = 0; m < M; ++m) {
        for (int g = 0; g < ng; ++g) {
            const uint16_t* xr = X + (size_t)m * ldx + (size_t)g * G;
            volatile float amax = 0.0f;
            for (int k = 0; k < G; ++k) {
                float xt = bf16_to_f32(xr[k]);
                if (tinv) xt = xt * tinv[g * G + k];
                float a = fabsf(xt);
                if (a > amax) amax = a;
            }
            float amax_c = amax > 0x1p-30f ? amax : 0x1p-30f;
            volatile float s = amax_c / 7.0f;
            volatile float inv = 1.0f / s;
            sx[(size_t)m * ng + g] = s;
            for (int k = 0; k < G; ++k) {
                float xt = bf16_to_f32(xr[k]);
                if (tinv) xt = xt * tinv[g * G + k];
                volatile float scaled = xt * inv;
                int qi = (int)nearbyintf(scaled);     /* default mode = round-half-even (R5) */
                if (qi > 7) qi = 7;
                if (qi < -7) qi = -7;
                q[(size_t)m * K + (size_t)g * G + k] = (int8_t)qi;
            }
        }
    }
}

/* ---- step 4: nibble pack / unpack (R10) ----------------------------------
 * byte j of a row = (q[2j] & 0xF) | ((q[2j+1] & 0xF) << 4), two's complement.
 */
void twq_oracle_pack_nibbles(const int8_t* q, int64_t rows, int K, uint8_t* out) {
    for (int64_t i = 0; i < rows; ++i)
        for (int j = 0; j < K / 2; ++j) {
            int lo = q[i * K + 2 * j] & 0xF;
            int hi = q[i * K + 2 * j + 1] & 0xF;
            out[i * (K / 2) + j] = (uint8_t)(lo | (hi << 4));
        }
}

static int nib_to_int(int n) { return n >= 8 ? n - 16 : n; }

void twq_oracle_unpack_nibbles(const uint8_t* p, int64_t rows, int K, int8_t* q) {
    for (int64_t i = 0; i < rows; ++i)
        for (int j = 0; j < K / 2; ++j) {
            uint8_t b = p[i * (K / 2) + j];
            q[i * K + 2 * j] = (int8_t)nib_to_int(b & 0xF);
            q[i * K + 2 * j + 1] = (int8_t)nib_to_int(b >> 4);
        }
}

/* ---- step 5: residual group products, exact integers ----------------------
 * PAPER.md L49-50 Eq. 2 (Q_X Q_W), L177 (integer accumulation), L193 (groups):
 *   P[m,g,n] = sum_{k in group g} qx[m,k] * qw[n,k]         (int64)
 * rows[i] selects token rows (NULL = all M rows, nrows = M).
 * Output P is [nrows, ng, N] int64.
 */
void twq_oracle_residual_P(const uint8_t* Xq, const uint8_t* R4, int M, int N, int K, int G,
                           const int* rows, int nrows, int64_t* P) {
    int ng = K / G;
    int8_t* qw = (int8_t*)malloc((size_t)N * K);
    twq_oracle_unpack_nibbles(R4, N, K, qw);
    (void)M;
#pragma omp parallel
    {
        int8_t* qx = (int8_t*)malloc((size_t)K);
#pragma omp for schedule(static) collapse(1)
        for (int i = 0; i < nrows; ++i) {
            int m = rows ? rows[i] : i;
            twq_oracle_unpack_nibbles(Xq + (size_t)m * (K / 2), 1, K, qx);
            for (int g = 0; g < ng; ++g)
                for (int n = 0; n < N; ++n) {
                    int64_t acc = 0;
                    for (int k = g * G; k < (g + 1) * G; ++k)
                        acc += (int64_t)qx[k] * (int64_t)qw[(size_t)n * K + k];
                    P[((size_t)i * ng + g) * N + n] = acc;
                }
        }
        free(qx);
    }
    free(qw);
}

/* ---- steps 5-8: whole forward ---------------------------------------------
 *   Yres[m,n] = sum_g (double)sx[m,g] * (double)sw[n,g] * (double)P[m,g,n]   (L181: fold scales)
 *   H[m,j]    = sum_k (double)X[m,k] * (double)L1[k,j]                        (Eq. 3 first term, stage 1)
 *   Ylr[m,n]  = sum_j H[m,j] * (double)L2[j,n]                               (stage 2; no intermediate rounding)
 *   Y[m,n]    = Yres + Ylr                                                   (L181: merge, one store)
 * Xq/sx are the quantizer outputs (steps 1-4); X is the raw BF16 activation
 * (the low-rank branch reads X untransformed: DESIGN.md reading R3).
 * sw, L1, L2 are FP16 bit patterns.  r may be 0 (plain W4A4).
 * Output Y is [nrows, N] double.  If P_out != NULL it receives [nrows, ng, N].
 * OpenMP over output channels n within a row, so M = 1 still uses the cores.
 */
void twq_oracle_forward(const uint16_t* X, int ldx, const uint8_t* Xq, const float* sx,
                        const uint8_t* R4, const uint16_t* sw,
                        const uint16_t* L1, const uint16_t* L2,
                        int M, int N, int K, int r, int G,
                        const int* rows, int nrows, double* Y, int64_t* P_out) {
    int ng = K / G;
    (void)M;
    int8_t* qw = (int8_t*)malloc((size_t)N * K);
    twq_oracle_unpack_nibbles(R4, N, K, qw);
    int8_t* qx = (int8_t*)malloc((size_t)K);
    double* H = (double*)malloc(sizeof(double) * (size_t)(r > 0 ? r : 1));
    for (int i = 0; i < nrows; ++i) {
        int m = rows ? rows[i] : i;
        twq_oracle_unpack_nibbles(Xq + (size_t)m * (K / 2), 1, K, qx);
        /* stage 1 of the low-rank branch */
        for (int j = 0; j < r; ++j) H[j] = 0.0;
        for (int k = 0; k < K; ++k) {
            double x = (double)bf16_to_f32(X[(size_t)m * ldx + k]);
            for (int j = 0; j < r; ++j) H[j] += x * fp16_to_f64(L1[(size_t)k * r + j]);
        }
#pragma omp parallel for schedule(static)
        for (int n = 0; n < N; ++n) {
            double yres = 0.0;
            for (int g = 0; g < ng; ++g) {
                int64_t acc = 0;
                for (int k = g * G; k < (g + 1) * G; ++k)
                    acc += (int64_t)qx[k] * (int64_t)qw[(size_t)n * K + k];
                if (P_out) P_out[((size_t)i * ng + g) * N + n] = acc;
                yres += (double)sx[(size_t)m * ng + g] * fp16_to_f64(sw[(size_t)n * ng + g]) * (double)acc;
            }
            double ylr = 0.0;
            for (int j = 0; j < r; ++j) ylr += H[j] * fp16_to_f64(L2[(size_t)j * N + n]);
            Y[(size_t)i * N + n] = yres + ylr;
        }
    }
    free(H);
    free(qx);
    free(qw);
}

/* ---- NEXT-1: the paper's own, fully 4-bit low-rank branch -------
 * PAPER.md L177-181 (section 4.3 "Fused two-stage low-rank pipeline", "On-the-fly scaling with a
 * single epilogue"), Eq. 4: Q(X)[Q(U)Q(V) + Q(R)].  Both low-rank factors are 4-bit with group
 * scales (L193) and the branch consumes the QUANTIZED activation ("quantizes the input activation
 * tile once and reuses it for both components", L179):
 *   P1[m,g,j] = sum_{k in g} qx[m,k] * qu[j,k]                exact int64 (first 4-bit GEMM, "int32 accumulation")
 *   H[m,j]    = sum_g sx[m,g] * su[j,g] * P1[m,g,j]           FP64 (the value of the INT32 accumulators with their scales)
 *   on-the-fly re-quantization (L181: "estimating an intermediate scale s_H from the INT32 accumulator and
 *   re-quantizing on the fly"); readings R18 / R19: the quantizer of Eq. 1 (L43-47) on float32(H), one
 *   scale per token and per group of Gr consecutive j (Gr = r for r <= 128, else 128), same FP32 operation order
 *   as the activation quantizer:
 *     a = max(max_{j in h} |H32[m,j]|, 2^-30);  sH[m,h] = a / 7.0f;  inv = 1.0f / sH;
 *     QH[m,j] = clamp(rint(H32[m,j] * inv), -7, 7)
 *   P2[m,h,n] = sum_{j in h} QH[m,j] * qv[n,j]                exact int64 (second 4-bit GEMM)
 *   Ylr[m,n]  = sum_h sH[m,h] * sv[n,h] * P2[m,h,n]           FP64
 *   Y         = Yres + Ylr                                    (single epilogue, L181)
 * U4 [r][K/2] and V4 [N][r/2] are nibble-packed like R4; su [r][K/G], sv [N][r/Gr] are FP16 bit patterns.
 * Optional outputs: H_out [nrows][r] (FP64), QH_out [nrows][r], sH_out [nrows][r/Gr].
 */
void twq_oracle_forward_q4lr(const uint8_t* Xq, const float* sx, const uint8_t* R4, const uint16_t* sw,
                             const uint8_t* U4, const uint16_t* su, const uint8_t* V4, const uint16_t* sv,
                             int M, int N, int K, int r, int G, int Gr, const int* rows, int nrows,
                             double* Y, double* H_out, int8_t* QH_out, float* sH_out) {
    int ng = K / G, nh = r / Gr;
    (void)M;
    int8_t* qw = (int8_t*)malloc((size_t)N * K);
    int8_t* qu = (int8_t*)malloc((size_t)r * K);
    int8_t* qv = (int8_t*)malloc((size_t)N * r);
    twq_oracle_unpack_nibbles(R4, N, K, qw);
    twq_oracle_unpack_nibbles(U4, r, K, qu);
    twq_oracle_unpack_nibbles(V4, N, r, qv);
    int8_t* qx = (int8_t*)malloc((size_t)K);
    double* H = (double*)malloc(sizeof(double) * (size_t)r);
    int8_t* QH = (int8_t*)malloc((size_t)r);
    float* sH = (float*)malloc(sizeof(float) * (size_t)nh);
    for (int i = 0; i < nrows; ++i) {
        int m = rows ? rows[i] : i;
        twq_oracle_unpack_nibbles(Xq + (size_t)m * (K / 2), 1, K, qx);
        /* first 4-bit GEMM + its scales */
        for (int j = 0; j < r; ++j) {
            double h = 0.0;
            for (int g = 0; g < ng; ++g) {
                int64_t acc = 0;
                for (int k = g * G; k < (g + 1) * G; ++k) acc += (int64_t)qx[k] * (int64_t)qu[(size_t)j * K + k];
                h += (double)sx[(size_t)m * ng + g] * fp16_to_f64(su[(size_t)j * ng + g]) * (double)acc;
            }
            H[j] = h;
            if (H_out) H_out[(size_t)i * r + j] = h;
        }
        /* on-the-fly re-quantization of H (Eq. 1 on float32(H), groups of Gr along r) */
        for (int h = 0; h < nh; ++h) {
            volatile float amax = 0.0f;
            for (int j = h * Gr; j < (h + 1) * Gr; ++j) {
                float a = fabsf((float)H[j]);
                if (a > amax) amax = a;
            }
            float amax_c = amax > 0x1p-30f ? amax : 0x1p-30f;
            volatile float s = amax_c / 7.0f;
            volatile float inv = 1.0f / s;
            sH[h] = s;
            if (sH_out) sH_out[(size_t)i * nh + h] = s;
            for (int j = h * Gr; j < (h + 1) * Gr; ++j) {
                volatile float scaled = (float)H[j] * inv;
                int qi = (int)nearbyintf(scaled);
                if (qi > 7) qi = 7;
                if (qi < -7) qi = -7;
                QH[j] = (int8_t)qi;
                if (QH_out) QH_out[(size_t)i * r + j] = (int8_t)qi;
            }
        }
#pragma omp parallel for schedule(static)
        for (int n = 0; n < N; ++n) {
            double yres = 0.0;
            for (int g = 0; g < ng; ++g) {
                int64_t acc = 0;
                for (int k = g * G; k < (g + 1) * G; ++k)
                    acc += (int64_t)qx[k] * (int64_t)qw[(size_t)n * K + k];
                yres += (double)sx[(size_t)m * ng + g] * fp16_to_f64(sw[(size_t)n * ng + g]) * (double)acc;
            }
            double ylr = 0.0;
            for (int h = 0; h < nh; ++h) {
                int64_t acc = 0;
                for (int j = h * Gr; j < (h + 1) * Gr; ++j) acc += (int64_t)QH[j] * (int64_t)qv[(size_t)n * r + j];
                ylr += (double)sH[h] * fp16_to_f64(sv[(size_t)n * nh + h]) * (double)acc;
            }
            Y[(size_t)i * N + n] = yres + ylr;
        }
    }
    free(sH); free(QH); free(H); free(qx); free(qv); free(qu); free(qw);
}

/* ---- output rounding: FP64 -> BF16 with ONE round-to-nearest-even ----------
 * (north_star: "BF16 output"; reading R11: exactly one rounding, at the store)
 */
void twq_oracle_round_bf16(const double* y, int64_t n, uint16_t* out) {
    for (int64_t i = 0; i < n; ++i) {
        double v = y[i];
        uint16_t sign = signbit(v) ? 0x8000 : 0;
        double a = fabs(v);
        if (isnan(v)) { out[i] = 0x7FC0; continue; }
        if (a == 0.0) { out[i] = sign; continue; }
        if (isinf(v)) { out[i] = sign | 0x7F80; continue; }
        int e = ilogb(a);
        if (e < -126) e = -126;                 /* BF16 subnormal quantum 2^-133 */
        double quantum = ldexp(1.0, e - 7);
        double rr = nearbyint(a / quantum) * quantum;   /* exact in double */
        if (rr >= ldexp(1.0, 128)) { out[i] = sign | 0x7F80; continue; }
        float f = (float)rr;                    /* exact: rr has <= 8 significant bits */
        uint32_t u;
        memcpy(&u, &f, 4);
        out[i] = sign | (uint16_t)(u >> 16);
    }
}

int twq_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
