/* gwo_oracle.c -- the ORACLE for the gwi hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, FP64, direct-convolution CPU implementation of what the hot path of arXiv 2201.11133
 * computes: the two-branch dilated-causal WaveNet-style detector, the 4-model ensemble
 * (PAPER.md:51, 136), ensemble averaging + threshold + width>=0.5 s trigger clustering (PAPER.md:102 as
 * restated by BASELINE.json) and time slides of L1 against H1.  The paper is silent on
 * every hyper-parameter; the readings A1..A31 taken are listed in DESIGN.md ("Readings") and cited below.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.
 * It shares no code with paper_2201_11133_b200/ (own file parser, own fp16 rounding, own everything).
 *
 * What is NOT here on purpose (it would not be "the definition written out"): streaming history reuse,
 * the split of the head's first conv across branches, tanh-for-sigmoid substitution, tiling, fusion.
 * The single liberty: loops are nested (out-channel, in-channel, tap, time) so the inner loop is a
 * contiguous axpy.  Per output element the additions still happen in the order  bias, then c-major /
 * tap-minor,  exactly as the formula reads.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 causality, P2 receptive field, P3 linearity/bias,
 * P4 dilation<->polyphase and shift, P5/P6 hand-worked examples (tests/golden), P7 closed forms,
 * P8 windowed==stream, P9 branch independence + slide reuse, P10 channel permutation, P11 batch
 * independence, P12 numpy.convolve cross-check, P13/P14 clustering worked example + brute force,
 * P16 sign pass-through closed form, P17 coincidence worked example + tuple brute force + invariances.
 * PARITY UNPINNED: the absolute probability values for the
 * random-weight configs have no external reference (no trained weights / LIGO data in this container).
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC gwo_oracle.c -o libgwo_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int n_branch, c_in, R, S, k, L, Hh;
    int *dil;          /* [L] */
    double **W_in;     /* [n_branch] -> [R][c_in] */
    double **b_in;     /* [n_branch] -> [R] */
    double **Wf, **bf, **Wg, **bg, **Wr, **br, **Ws, **bs; /* [n_branch*L] */
    double *W1, *b1, *W2; /* [Hh][n_branch*S], [Hh], [Hh] */
    double b2;
} gwo_model;

typedef struct {
    int32_t slide;
    int32_t model_mask;
    int64_t start, end; /* [start, end) in samples, global index */
    double peak_p, mean_p;
} gwo_trigger;

/* ---- fp16 rounding (own implementation; FP16 mode rounds weights and inputs, reading A14 / C.2) ------- */
/* float -> IEEE binary16 with round-to-nearest-even -> double.  Overflow goes to +-inf like the hardware. */
double gwo_round_half(double v)
{
    float f = (float)v;
    uint32_t u; memcpy(&u, &f, 4);
    uint32_t sign = u >> 31, ex = (u >> 23) & 0xff, man = u & 0x7fffff;
    double s = sign ? -1.0 : 1.0;
    if (ex == 0xff) return man ? NAN : s * INFINITY;
    int e = (int)ex - 127;                       /* unbiased exponent of the float */
    if (ex == 0) return s * 0.0;                 /* float subnormal: far below half's smallest subnormal */
    if (e < -25) return s * 0.0;                 /* below half of the smallest half subnormal (2^-24) */
    uint64_t sig = (uint64_t)(man | 0x800000);   /* 24-bit significand, value = sig * 2^(e-23) */
    int shift;                                    /* number of low bits to drop */
    if (e >= -14) shift = 13;                    /* normal half: keep 11 significant bits */
    else shift = 13 + (-14 - e);                 /* subnormal half: fixed quantum 2^-24 */
    uint64_t keep = sig >> shift;
    uint64_t rem = sig & (((uint64_t)1 << shift) - 1);
    uint64_t halfway = (uint64_t)1 << (shift - 1);
    if (rem > halfway || (rem == halfway && (keep & 1))) keep++;
    double r = ldexp((double)keep, e - 23 + shift);
    if (r >= 65520.0) return s * INFINITY;       /* 65504 is the max finite half; 65520 rounds up to inf */
    return s * r;
}

/* ---- model file (GWIM v1; layout documented in gwsynth/modelfile.py and DESIGN.md) --------------------- */
static double *read_tensor(FILE *f, size_t n, int round_fp16)
{
    float *tmp = (float *)malloc(n * sizeof(float));
    double *d = (double *)malloc(n * sizeof(double));
    if (!tmp || !d || fread(tmp, sizeof(float), n, f) != n) { free(tmp); free(d); return NULL; }
    for (size_t i = 0; i < n; i++) d[i] = round_fp16 ? gwo_round_half((double)tmp[i]) : (double)tmp[i];
    free(tmp);
    return d;
}

void gwo_free_model(gwo_model *m)
{
    if (!m) return;
    int nb = m->n_branch, nl = m->n_branch * m->L;
    if (m->W_in) for (int b = 0; b < nb; b++) { free(m->W_in[b]); free(m->b_in[b]); }
    double ***per_layer[] = {&m->Wf, &m->bf, &m->Wg, &m->bg, &m->Wr, &m->br, &m->Ws, &m->bs};
    for (int a = 0; a < 8; a++) if (*per_layer[a]) { for (int i = 0; i < nl; i++) free((*per_layer[a])[i]); free(*per_layer[a]); }
    free(m->W_in); free(m->b_in); free(m->W1); free(m->b1); free(m->W2); free(m->dil); free(m);
}

/* returns 0 on success, 2 = cannot open/short file, 3 = bad format */
int gwo_load_model(const char *path, int round_fp16, gwo_model **out)
{
    FILE *f = fopen(path, "rb");
    if (!f) return 2;
    char magic[4]; int32_t hdr[9];
    if (fread(magic, 1, 4, f) != 4 || fread(hdr, 4, 9, f) != 9) { fclose(f); return 2; }
    if (memcmp(magic, "GWIM", 4) != 0 || hdr[0] != 1 || hdr[8] != 0) { fclose(f); return 3; }
    gwo_model *m = (gwo_model *)calloc(1, sizeof(gwo_model));
    m->n_branch = hdr[1]; m->c_in = hdr[2]; m->R = hdr[3]; m->S = hdr[4]; m->k = hdr[5]; m->L = hdr[6]; m->Hh = hdr[7];
    if (m->n_branch < 1 || m->c_in < 1 || m->R < 1 || m->S < 1 || m->k < 1 || m->L < 1 || m->Hh < 1 || m->L > 4096) { free(m); fclose(f); return 3; }
    m->dil = (int *)malloc(sizeof(int) * m->L);
    int32_t *d32 = (int32_t *)malloc(4 * m->L);
    if (fread(d32, 4, m->L, f) != (size_t)m->L) { free(d32); gwo_free_model(m); fclose(f); return 2; }
    for (int i = 0; i < m->L; i++) { m->dil[i] = d32[i]; if (d32[i] < 1) { free(d32); gwo_free_model(m); fclose(f); return 3; } }
    free(d32);
    int nb = m->n_branch, nl = nb * m->L, R = m->R, S = m->S, k = m->k;
    m->W_in = (double **)calloc(nb, sizeof(double *)); m->b_in = (double **)calloc(nb, sizeof(double *));
    double ***per_layer[] = {&m->Wf, &m->bf, &m->Wg, &m->bg, &m->Wr, &m->br, &m->Ws, &m->bs};
    for (int a = 0; a < 8; a++) *per_layer[a] = (double **)calloc(nl, sizeof(double *));
    int ok = 1;
    for (int b = 0; b < nb && ok; b++) {
        ok = ok && (m->W_in[b] = read_tensor(f, (size_t)R * m->c_in, round_fp16));
        ok = ok && (m->b_in[b] = read_tensor(f, R, round_fp16));
        for (int i = 0; i < m->L && ok; i++) {
            int q = b * m->L + i;
            ok = ok && (m->Wf[q] = read_tensor(f, (size_t)R * R * k, round_fp16));
            ok = ok && (m->bf[q] = read_tensor(f, R, round_fp16));
            ok = ok && (m->Wg[q] = read_tensor(f, (size_t)R * R * k, round_fp16));
            ok = ok && (m->bg[q] = read_tensor(f, R, round_fp16));
            ok = ok && (m->Wr[q] = read_tensor(f, (size_t)R * R, round_fp16));
            ok = ok && (m->br[q] = read_tensor(f, R, round_fp16));
            ok = ok && (m->Ws[q] = read_tensor(f, (size_t)S * R, round_fp16));
            ok = ok && (m->bs[q] = read_tensor(f, S, round_fp16));
        }
    }
    double *b2 = NULL;
    ok = ok && (m->W1 = read_tensor(f, (size_t)m->Hh * nb * S, round_fp16));
    ok = ok && (m->b1 = read_tensor(f, m->Hh, round_fp16));
    ok = ok && (m->W2 = read_tensor(f, m->Hh, round_fp16));
    ok = ok && (b2 = read_tensor(f, 1, round_fp16));
    if (ok) { m->b2 = b2[0]; }
    free(b2);
    int trailing = ok ? (fgetc(f) != EOF) : 0;
    fclose(f);
    if (!ok) { gwo_free_model(m); return 2; }
    if (trailing) { gwo_free_model(m); return 3; }
    *out = m;
    return 0;
}

void gwo_model_info(const gwo_model *m, int32_t *n_branch, int32_t *c_in, int32_t *R, int32_t *S, int32_t *k,
                    int32_t *L, int32_t *Hh, int32_t *receptive_field)
{
    long sum = 0; for (int i = 0; i < m->L; i++) sum += m->dil[i];
    *n_branch = m->n_branch; *c_in = m->c_in; *R = m->R; *S = m->S; *k = m->k; *L = m->L; *Hh = m->Hh;
    *receptive_field = (int32_t)(1 + (long)(m->k - 1) * sum);      /* R_f = 1 + (k-1) sum d_i  (reading A3) */
}

/* ---- one causal dilated convolution (DESIGN.md C.1 step 2; readings A4 padding, A5 tap order) ----------
 * y[o][t] = b[o] + sum_c sum_j W[o][c][j] * x[c][t - (k-1-j)*d],   reads at index < 0 return 0.
 * x: [Cin][T], y: [Cout][T], W: [Cout][Cin][k].  Tap j = k-1 is the current sample.                       */
void gwo_conv1d_causal(const double *x, int Cin, int Cout, int k, int d, const double *W, const double *b,
                       long T, double *y)
{
    for (int o = 0; o < Cout; o++) {
        double *yo = y + (size_t)o * T;
        for (long t = 0; t < T; t++) yo[t] = b ? b[o] : 0.0;
        for (int c = 0; c < Cin; c++) {
            const double *xc = x + (size_t)c * T;
            for (int j = 0; j < k; j++) {
                double w = W[((size_t)o * Cin + c) * k + j];
                long back = (long)(k - 1 - j) * d;       /* how far in the past this tap reads */
                for (long t = back; t < T; t++) yo[t] += w * xc[t - back];   /* t < back reads padding = 0 */
            }
        }
    }
}

/* ---- one branch (C.1 steps 1-3).  x: [c_in][T].  u: [S][T].  h_dump (optional): [L+1][R][T] ----------- */
void gwo_branch(const gwo_model *m, int b, const double *x, long T, double *u, double *h_dump)
{
    int R = m->R, S = m->S, k = m->k;
    size_t RT = (size_t)R * T, ST = (size_t)S * T;
    double *h = (double *)malloc(RT * 8), *f = (double *)malloc(RT * 8), *g = (double *)malloc(RT * 8);
    double *z = (double *)malloc(RT * 8), *s = (double *)malloc(ST * 8), *r = (double *)malloc(RT * 8);
    /* 1. lift: h0[r][t] = b_in[r] + sum_c W_in[r][c] x[c][t]   (1x1 conv, no activation; reading A3) */
    gwo_conv1d_causal(x, m->c_in, R, 1, 1, m->W_in[b], m->b_in[b], T, h);
    if (h_dump) memcpy(h_dump, h, RT * 8);
    for (size_t i = 0; i < ST; i++) u[i] = 0.0;                /* skip sum, plain sum over blocks (A9) */
    for (int i = 0; i < m->L; i++) {
        int q = b * m->L + i, d = m->dil[i];
        /* 2. f, g = causal dilated convs of the block input (A6: separate Wf, Wg) */
        gwo_conv1d_causal(h, R, R, k, d, m->Wf[q], m->bf[q], T, f);
        gwo_conv1d_causal(h, R, R, k, d, m->Wg[q], m->bg[q], T, g);
        /*    z = tanh(f) * sigma(g) */
        for (size_t e = 0; e < RT; e++) z[e] = tanh(f[e]) * (1.0 / (1.0 + exp(-g[e])));
        /*    skip_i = bs + Ws z ;  h_i = h_{i-1} + br + Wr z     (A7: both 1x1 convs on z with bias) */
        gwo_conv1d_causal(z, R, S, 1, 1, m->Ws[q], m->bs[q], T, s);
        for (size_t e = 0; e < ST; e++) u[e] += s[e];
        gwo_conv1d_causal(z, R, R, 1, 1, m->Wr[q], m->br[q], T, r);
        for (size_t e = 0; e < RT; e++) h[e] = h[e] + r[e];
        if (h_dump) memcpy(h_dump + (size_t)(i + 1) * RT, h, RT * 8);
    }
    /* 3. branch output u = ReLU(sum_i skip_i) */
    for (size_t e = 0; e < ST; e++) u[e] = u[e] > 0.0 ? u[e] : 0.0;
    free(h); free(f); free(g); free(z); free(s); free(r);
}

/* ---- head (C.1 steps 4-5; reading A10 concat H1 first, A11 two 1x1 convs, ReLU, single-logit sigmoid) ---
 * ucat: n_branch pointers, each [S][T].  lag[b]: branch b's feature is read at (t - lag[b]) mod T
 * (lag = 0 everywhere for the ordinary forward pass; the slide definition A24 uses lag[1] = k*fs).        */
static void head_eval(const gwo_model *m, const double *const *ucat, const long *lag, long T, double *p)
{
    int S = m->S, nb = m->n_branch, Hh = m->Hh;
    for (long t = 0; t < T; t++) {
        double y = m->b2;
        for (int a = 0; a < Hh; a++) {
            double v = m->b1[a];
            for (int b = 0; b < nb; b++) {
                long tb = t;
                if (lag && lag[b]) { tb = (t - lag[b]) % T; if (tb < 0) tb += T; }
                for (int q = 0; q < S; q++) v += m->W1[(size_t)a * nb * S + (size_t)b * S + q] * ucat[b][(size_t)q * T + tb];
            }
            v = v > 0.0 ? v : 0.0;
            y += m->W2[a] * v;
        }
        p[t] = 1.0 / (1.0 + exp(-y));
    }
}

/* ---- whole model on one sequence.  x: [n_branch*c_in][T] planar (H1 channels first).  p: [T].
 *      u_out (optional): [n_branch][S][T] branch features.                                              */
void gwo_forward(const gwo_model *m, const double *x, long T, double *p, double *u_out)
{
    int nb = m->n_branch, S = m->S;
    double *u = u_out ? u_out : (double *)malloc((size_t)nb * S * T * 8);
    const double **up = (const double **)malloc(nb * sizeof(double *));
    for (int b = 0; b < nb; b++) {
        gwo_branch(m, b, x + (size_t)b * m->c_in * T, T, u + (size_t)b * S * T, NULL);
        up[b] = u + (size_t)b * S * T;
    }
    head_eval(m, up, NULL, T, p);
    free(up);
    if (!u_out) free(u);
}

/* ---- window API (the paper's tensor contract): x [B][T][C] channels-last, p [B][T].
 *      Each window is evaluated independently with zero history (reading A15 "window API").              */
void gwo_infer_windows(const gwo_model *m, const double *x, long B, long T, double *p)
{
    int C = m->n_branch * m->c_in;
#pragma omp parallel for schedule(dynamic, 1)
    for (long w = 0; w < B; w++) {
        double *xp = (double *)malloc((size_t)C * T * 8);
        for (long t = 0; t < T; t++) for (int c = 0; c < C; c++) xp[(size_t)c * T + t] = x[((size_t)w * T + t) * C + c];
        gwo_forward(m, xp, T, p + (size_t)w * T, NULL);
        free(xp);
    }
}

/* ---- stream: p_stream[t], t in [0,N), is gwo_forward over the whole stream with T = N (zero history only
 *      at t = 0).  To bound memory it is evaluated on segments [s0, s1) extended backwards by R_f - 1
 *      samples; every layer of a segment computes the very same sums as the whole-stream pass for
 *      t >= s0 (values in the discarded halo differ).  tests pin: segmented == unsegmented bit-for-bit.
 *      x: [C][N] planar.  u_out optional [n_branch][S][N].                                              */
void gwo_stream(const gwo_model *m, const double *x, long N, long seg, double *p, double *u_out)
{
    int C = m->n_branch * m->c_in, nb = m->n_branch, S = m->S;
    long sum = 0; for (int i = 0; i < m->L; i++) sum += m->dil[i];
    long halo = (long)(m->k - 1) * sum;
    if (seg <= 0 || seg > N) seg = N;
    long nseg = (N + seg - 1) / seg;
#pragma omp parallel for schedule(dynamic, 1)
    for (long q = 0; q < nseg; q++) {
        long s0 = q * seg, s1 = s0 + seg < N ? s0 + seg : N;
        long a0 = s0 - halo > 0 ? s0 - halo : 0, Tl = s1 - a0, off = s0 - a0;
        double *xl = (double *)malloc((size_t)C * Tl * 8), *pl = (double *)malloc((size_t)Tl * 8);
        double *ul = (double *)malloc((size_t)nb * S * Tl * 8);
        for (int c = 0; c < C; c++) memcpy(xl + (size_t)c * Tl, x + (size_t)c * N + a0, (size_t)Tl * 8);
        gwo_forward(m, xl, Tl, pl, ul);
        memcpy(p + s0, pl + off, (size_t)(s1 - s0) * 8);
        if (u_out) for (int b = 0; b < nb; b++) for (int s = 0; s < S; s++)
            memcpy(u_out + ((size_t)b * S + s) * N + s0, ul + ((size_t)b * S + s) * Tl + off, (size_t)(s1 - s0) * 8);
        free(xl); free(pl); free(ul);
    }
}

/* ---- slide k (reading A24): p_k[t] = head(u_H1[.][t], u_L1[.][(t - lag) mod N]); u: [n_branch][S][N];
 *      every branch b >= 1 is delayed by `lag` samples, branch 0 (H1) is the time reference.            */
void gwo_head_slide(const gwo_model *m, const double *u, long N, long lag, double *p)
{
    int nb = m->n_branch, S = m->S;
    const double **up = (const double **)malloc(nb * sizeof(double *));
    long *lg = (long *)calloc(nb, sizeof(long));
    for (int b = 0; b < nb; b++) { up[b] = u + (size_t)b * S * N; lg[b] = b ? lag : 0; }
    head_eval(m, up, lg, N, p);
    free(up); free(lg);
}

/* ---- ensemble mean (reading A18): arithmetic mean of probabilities in model order -------------------- */
void gwo_ensemble_mean(const double *const *p, int M, long N, double *pbar)
{
    for (long t = 0; t < N; t++) { double s = p[0][t]; for (int j = 1; j < M; j++) s += p[j][t]; pbar[t] = s / (double)M; }
}
/* tier T1: the interface on materialised FP32 arrays fixes the FP32 expression (((p0+p1)+p2)+...)/(float)M */
void gwo_ensemble_mean_f32(const float *const *p, int M, long N, float *pbar)
{
    for (long t = 0; t < N; t++) {
        volatile float s = p[0][t];
        for (int j = 1; j < M; j++) s = s + p[j][t];
        pbar[t] = s / (float)M;
    }
}

/* ---- triggers (readings A19 strict >, A20 run length >= L_min, A21 edges, A22 record) ------------------
 * a[t] = (pbar[t] > theta); maximal runs [s,e) of a = 1 with e - s >= L_min are emitted in order of s.
 * Runs touching either end of [0,N) count with their truncated length.  t0 is added to start/end.
 * pm (optional, M pointers): model_mask bit j = model j has pm[j][t] > theta for some t in the run.
 * Returns the total number of qualifying runs; writes at most cap records.                              */
long gwo_triggers(const double *pbar, long N, double theta, long Lmin, int slide, long t0,
                  const double *const *pm, int M, gwo_trigger *out, long cap)
{
    long count = 0, t = 0;
    while (t < N) {
        if (!(pbar[t] > theta)) { t++; continue; }
        long s = t;
        double peak = pbar[t], sum = 0.0;
        int32_t mask = 0;
        while (t < N && pbar[t] > theta) {
            if (pbar[t] > peak) peak = pbar[t];
            sum += pbar[t];
            if (pm) for (int j = 0; j < M && j < 31; j++) if (pm[j][t] > theta) mask |= (1 << j);
            t++;
        }
        if (t - s >= Lmin) {
            if (count < cap) {
                out[count].slide = slide; out[count].model_mask = mask;
                out[count].start = s + t0; out[count].end = t + t0;
                out[count].peak_p = peak; out[count].mean_p = sum / (double)(t - s);
            }
            count++;
        }
    }
    return count;
}

/* ---- all-model coincidence of per-model triggers ("Triggers that were reported by all AI models in
 * the ensemble, and which were coincident within a time window of 0.5 seconds were flagged as gravitational wave
 * events"; reading A34) ------------------------------------------------------------------------------------------
 * ends[m][i], i < n[m]: merger-time estimates (trigger ends) of model m, any order.
 * A time a is an ANCHOR iff a is one of the ends and every model has an end in [a, a + W].
 * Anchors are sorted; a new event starts at an anchor that is more than W after the previous anchor.
 * Event: t_first = its first anchor, t_last = the largest end (any model) in [t_first, last anchor + W],
 * n_triggers = number of ends (all models) in [t_first, last anchor + W].  Plain O(n^2) scans.           */
typedef struct { int64_t t_first, t_last; int32_t n_triggers, slide; } gwo_event;

long gwo_coincidence(const long *const *ends, const int *n, int M, long W, int slide, gwo_event *out, long cap)
{
    long na = 0, tot = 0;
    for (int m = 0; m < M; m++) tot += n[m];
    long *anch = (long *)malloc((size_t)(tot > 0 ? tot : 1) * sizeof(long));
    for (int m = 0; m < M; m++)
        for (int i = 0; i < n[m]; i++) {
            long a = ends[m][i];
            int all = 1;
            for (int q = 0; q < M && all; q++) {
                int found = 0;
                for (int j = 0; j < n[q]; j++) if (ends[q][j] >= a && ends[q][j] <= a + W) found = 1;
                all = found;
            }
            if (all) anch[na++] = a;
        }
    for (long i = 1; i < na; i++) {                      /* insertion sort */
        long v = anch[i], j = i - 1;
        while (j >= 0 && anch[j] > v) { anch[j + 1] = anch[j]; j--; }
        anch[j + 1] = v;
    }
    long count = 0, i = 0;
    while (i < na) {
        long first = anch[i], last = anch[i];
        while (i + 1 < na && anch[i + 1] - last <= W) { i++; last = anch[i]; }
        i++;
        long tl = first; int nt = 0;
        for (int m = 0; m < M; m++)
            for (int j = 0; j < n[m]; j++)
                if (ends[m][j] >= first && ends[m][j] <= last + W) { nt++; if (ends[m][j] > tl) tl = ends[m][j]; }
        if (count < cap) { out[count].t_first = first; out[count].t_last = tl; out[count].n_triggers = nt; out[count].slide = slide; }
        count++;
    }
    free(anch);
    return count;
}

int gwo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- the paper's post-processing rule as stated: SciPy's find_peaks with a height and a width condition ------------
 * PAPER.md:53 ("post-processed it with the find_peaks algorithm, a SciPy's off-the-shelve tool"), PAPER.md:102 ("uses the
 * find_peaks algorithm to identity peaks whose width is at least 0.5 seconds long ... height in our find_peaks
 * algorithms").  find_peaks(x, height=h, width=w) is a public, fully defined procedure; it is restated here step by
 * step (SciPy reference guide, scipy.signal.find_peaks / peak_prominences / peak_widths, default wlen = None and
 * rel_height = 0.5):
 *  1. local maxima: i is a peak iff x[i-1] < x[i] and x[i] > x[i+1]; a flat top x[i] = ... = x[j] with x[i-1] < x[i] and
 *     x[j] > x[j+1] counts once, at floor((i + j) / 2); the first and the last sample are never peaks (a flat top that
 *     reaches either end of the array is not one).
 *  2. height: keep peaks with x[p] >= h.
 *  3. prominence of p: walk left from p while x[i] <= x[p] (stop at the array start), left_min = smallest value met;
 *     likewise to the right; prominence = x[p] - max(left_min, right_min).
 *  4. width of p at rel_height 0.5: level = x[p] - prominence / 2; walk left from p while level < x[i] (not past the
 *     position of left_min), the crossing is interpolated linearly between that sample and the one after it; likewise
 *     to the right; width = right crossing - left crossing (in samples).
 *  5. keep peaks with width >= w.  Output sorted by position.
 * TEST INFRASTRUCTURE like everything in this file; pinned against scipy.signal.find_peaks in tests/test_oracle_peaks.py. */
typedef struct { int64_t index; double height, prominence, width, left_ip, right_ip; } gwo_peak;

long gwo_find_peaks(const double *x, long N, double hmin, double wmin, gwo_peak *out, long cap)
{
    long count = 0;
    long i = 1;
    while (i < N - 1) {
        if (x[i - 1] < x[i]) {
            long j = i;                                   /* end of the flat top that starts at i */
            while (j < N - 1 && x[j + 1] == x[i]) j++;
            if (j < N - 1 && x[j + 1] < x[i]) {
                long p = (i + j) / 2;
                if (x[p] >= hmin) {
                    /* step 3 */
                    double lmin = x[p], rmin = x[p];
                    long lb = p, rb = p;
                    for (long k = p; k >= 0 && x[k] <= x[p]; k--) if (x[k] < lmin) { lmin = x[k]; lb = k; }
                    for (long k = p; k < N && x[k] <= x[p]; k++) if (x[k] < rmin) { rmin = x[k]; rb = k; }
                    double prom = x[p] - (lmin > rmin ? lmin : rmin);
                    /* step 4 */
                    double level = x[p] - prom * 0.5;
                    long k = p;
                    while (lb < k && level < x[k]) k--;
                    double lip = (double)k;
                    if (x[k] < level) lip += (level - x[k]) / (x[k + 1] - x[k]);
                    k = p;
                    while (k < rb && level < x[k]) k++;
                    double rip = (double)k;
                    if (x[k] < level) rip -= (level - x[k]) / (x[k - 1] - x[k]);
                    double width = rip - lip;
                    if (width >= wmin) {
                        if (count < cap) {
                            out[count].index = p; out[count].height = x[p]; out[count].prominence = prom;
                            out[count].width = width; out[count].left_ip = lip; out[count].right_ip = rip;
                        }
                        count++;
                    }
                }
            }
            i = j + 1;
        } else {
            i++;
        }
    }
    return count;
}
