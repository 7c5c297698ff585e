/*
 * hypic_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64, token-by-token CPU oracle for the linear-attention hot path of HYPIC
 * (arxiv/paper_2607_01299, contribution C1).  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.  It shares no code, header, table or
 * helper with the CUDA path under paper_2607_01299_b200/csrc/, and neither includes the other.
 *
 * What it computes (row convention of BASELINE.json:north_star; the paper writes the transpose,
 * see DESIGN.md reading A1):
 *
 *   state  S in R^{dv x dk},  transition accumulator  T in R^{dk x dk}
 *   token step (Eq. 2, with Table 1's dense family):
 *       paper:  S_i = T_i S_{i-1} + u_i,  T_i = g_i (I - beta_i k_i k_i^T)      (GDN, scalar gate)
 *                                         T_i = (I - beta_i k_i k_i^T) diag(g_i) (KDA, per-channel gate)
 *               u_i = beta_i k_i v_i^T
 *       here (transposed):  S <- S diag(a_t);  S <- S + beta_t (v_t - S k_t) k_t^T,   a_t = exp(g_t)
 *   segment-cumulative transition (Eq. 4): T_C = prod_{t in C} T_t, ordered
 *       (prod_{i=n}^{1} = T_n ... T_1 in the paper's left-multiplying convention, so the
 *       first token is the LEFTMOST factor in the row convention):  T <- T diag(a_t) (I - beta_t k_t k_t^T)
 *   zero-start end-state: E = S after the segment's tokens, started from S = 0
 *   composition (Eq. 4, Eq. 6):  S <- S T_i + E_i, i in list order
 *   scalar / diagonal families (Table 1, Table 3): S <- S diag(a_t) + v_t k_t^T,
 *       T_C = prod a_t kept as one scalar or a dk-vector, composition S <- S diag(t_i) + E_i  (hypic_oracle_diag_*)
 *   seam-window step (Fig. 8): token steps from a given running state, with the read-out
 *       of PAPER.md:86-90 (Eq. 2) after each step:  paper o_i = q_i^T S_i;  here o_t = S_t q_t
 *
 * There is no chunking, blocking, fusion or reordering here: one token at a time, one row at a time.
 * All pins are in tests/test_oracle_pins.py (P1..P10, W1..W4, D1..D5 and R1..R3 of DESIGN.md); no function here is "parity unpinned".
 *
 * Build: gcc -O3 -march=native -fopenmp -shared -fPIC hypic_oracle.c -o libhypic_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define HYPIC_ORACLE_GATE_SCALAR 0
#define HYPIC_ORACLE_GATE_CHANNEL 1

int hypic_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void hypic_oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/*
 * One token applied to a row-block M [rows x dk] (M is S with rows = dv, or T with rows = dk).
 * PAPER.md:84 (Eq. 2) + PAPER.md:61 (Table 1, GDN / KDA rows), transposed:
 *     M <- M diag(a);   M <- M + beta (w - M k) k^T
 * where w = v_t for the state S (write term u_t = beta k v^T, reading G1) and w = 0 for T
 * (T has no write term: it is the pure product of the T_t).
 * a points at dk decay factors (already exp'd); for the scalar gate all dk entries are equal.
 */
static void token_step(double* M, int rows, int dk, const double* a, const double* kt,
                       const double* w /* rows values, or NULL for zeros */, double beta) {
  for (int i = 0; i < rows; ++i) {
    double* row = M + (size_t)i * dk;
    double dot = 0.0;
    for (int c = 0; c < dk; ++c) {
      row[c] *= a[c];       /* decay first (reading A3) ... */
      dot += row[c] * kt[c]; /* ... then read the decayed state along k_t */
    }
    const double wi = w ? w[i] : 0.0;
    const double coef = beta * (wi - dot);
    for (int c = 0; c < dk; ++c) row[c] += coef * kt[c];
  }
}

/*
 * Scan one (segment, head): tokens [t0, t1) of head h.  S (dv x dk) and/or T (dk x dk) are updated in
 * place, whichever is non-NULL.  Inputs are the packed arrays of the C ABI:
 * k:[Ttot,H,dk], v:[Ttot,H,dv], g:[Ttot,H] (scalar gate) or [Ttot,H,dk] (per-channel gate), beta:[Ttot,H],
 * all float32 holding the exact input values (bf16 inputs are widened by the caller, which is exact).
 */
static void scan_unit(const float* k, const float* v, const float* g, const float* beta, int t0, int t1,
                      int h, int H, int dk, int dv, int gate, double* S, double* T) {
  double* a = (double*)malloc(sizeof(double) * (size_t)dk);
  double* kt = (double*)malloc(sizeof(double) * (size_t)dk);
  double* vt = (double*)malloc(sizeof(double) * (size_t)dv);
  for (int t = t0; t < t1; ++t) {
    const size_t th = (size_t)t * H + h;
    for (int c = 0; c < dk; ++c) kt[c] = (double)k[th * dk + c];
    for (int i = 0; i < dv; ++i) vt[i] = (double)v[th * dv + i];
    if (gate == HYPIC_ORACLE_GATE_CHANNEL) {
      for (int c = 0; c < dk; ++c) a[c] = exp((double)g[th * dk + c]); /* alpha = exp(g), reading A2 */
    } else {
      const double as = exp((double)g[th]);
      for (int c = 0; c < dk; ++c) a[c] = as;
    }
    const double b = (double)beta[th];
    if (S) token_step(S, dv, dk, a, kt, vt, b);
    if (T) token_step(T, dk, dk, a, kt, NULL, b);
  }
  free(a);
  free(kt);
  free(vt);
}

/*
 * hypic_oracle_segment_encode: for every segment s and head h, the zero-start end-state
 * E[s,h] (dv x dk; "S_{C|0}") and the segment-cumulative transition T[s,h] (dk x dk;
 * PAPER.md:120 "T_C := prod_{t in C} T_t").  A zero-length segment gives E = 0, T = I.
 * E:[n_seg,H,dv,dk], T:[n_seg,H,dk,dk] row-major doubles.  Either output may be NULL.
 * Returns 0, or 1 on a bad argument.
 */
int hypic_oracle_segment_encode(const float* k, const float* v, const float* g, const float* beta,
                                const int32_t* cu_seqlens, int n_seg, int H, int dk, int dv, int gate,
                                double* E, double* T) {
  if (n_seg < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_seqlens) return 1;
  if (gate != HYPIC_ORACLE_GATE_SCALAR && gate != HYPIC_ORACLE_GATE_CHANNEL) return 1;
  const long n_units = (long)n_seg * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int s = (int)(u / H), h = (int)(u % H);
    double* Eu = E ? E + (size_t)u * dv * dk : NULL;
    double* Tu = T ? T + (size_t)u * dk * dk : NULL;
    if (Eu) memset(Eu, 0, sizeof(double) * (size_t)dv * dk); /* S_0 = 0 */
    if (Tu) {
      memset(Tu, 0, sizeof(double) * (size_t)dk * dk);
      for (int c = 0; c < dk; ++c) Tu[(size_t)c * dk + c] = 1.0; /* empty product = I */
    }
    scan_unit(k, v, g, beta, cu_seqlens[s], cu_seqlens[s + 1], h, H, dk, dv, gate, Eu, Tu);
  }
  return 0;
}

/*
 * hypic_oracle_sequential: the thing composition must equal (Insight 1: composing
 * "recovers the exact end-state").  For each request r and head h, run the token recurrence (Eq. 2) over the
 * tokens [cu_tokens[r], cu_tokens[r+1]) starting from S_in[r,h] (NULL = zeros); no segment structure at all.
 * S_in, S_out: [R,H,dv,dk] doubles.
 */
int hypic_oracle_sequential(const double* S_in, const float* k, const float* v, const float* g,
                            const float* beta, const int32_t* cu_tokens, int R, int H, int dk, int dv,
                            int gate, double* S_out) {
  if (R < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_tokens || !S_out) return 1;
  if (gate != HYPIC_ORACLE_GATE_SCALAR && gate != HYPIC_ORACLE_GATE_CHANNEL) return 1;
  const long n_units = (long)R * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int r = (int)(u / H), h = (int)(u % H);
    double* Su = S_out + (size_t)u * dv * dk;
    if (S_in)
      memcpy(Su, S_in + (size_t)u * dv * dk, sizeof(double) * (size_t)dv * dk);
    else
      memset(Su, 0, sizeof(double) * (size_t)dv * dk);
    scan_unit(k, v, g, beta, cu_tokens[r], cu_tokens[r + 1], h, H, dk, dv, gate, Su, NULL);
  }
  return 0;
}

/*
 * hypic_oracle_seam_window: the seam-window step of PAPER.md:232-234 (section 4.3, Fig. 8): a few uncached tokens
 * are run through a linear layer on the fly, from the running state in front of them, and their per-token outputs are
 * emitted.  For each request r and head h: S = S_in[r,h] (NULL = zeros); for every token t of
 * [cu_tokens[r], cu_tokens[r+1]): one token step (Eq. 2, as in hypic_oracle_sequential), then the read-out
 * of PAPER.md:86-90 (Eq. 2, "o_i = q_i^T S_i") in the row convention:  o_t = S_t q_t  (a dv-vector; the state AFTER
 * token t's update is read).  q:[Ttot,H,dk] float32, o:[Ttot,H,dv] doubles (rows of tokens outside every request are
 * left untouched), S_out:[R,H,dv,dk] doubles.  Returns 0, or 1 on a bad argument.
 */
int hypic_oracle_seam_window(const double* S_in, const float* q, const float* k, const float* v, const float* g,
                             const float* beta, const int32_t* cu_tokens, int R, int H, int dk, int dv, int gate,
                             double* S_out, double* o) {
  if (R < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_tokens || !S_out || !o) return 1;
  if (gate != HYPIC_ORACLE_GATE_SCALAR && gate != HYPIC_ORACLE_GATE_CHANNEL) return 1;
  const long n_units = (long)R * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int r = (int)(u / H), h = (int)(u % H);
    double* Su = S_out + (size_t)u * dv * dk;
    if (S_in)
      memcpy(Su, S_in + (size_t)u * dv * dk, sizeof(double) * (size_t)dv * dk);
    else
      memset(Su, 0, sizeof(double) * (size_t)dv * dk);
    for (int t = cu_tokens[r]; t < cu_tokens[r + 1]; ++t) {
      scan_unit(k, v, g, beta, t, t + 1, h, H, dk, dv, gate, Su, NULL); /* one token step */
      const size_t th = (size_t)t * H + h;
      for (int i = 0; i < dv; ++i) {
        double acc = 0.0;
        for (int c = 0; c < dk; ++c) acc += Su[(size_t)i * dk + c] * (double)q[th * dk + c];
        o[th * dv + i] = acc;
      }
    }
  }
  return 0;
}

/*
 * Scalar and diagonal families of PAPER.md:57-61 (Table 1): T_i = a_i I (RetNet / Lightning-2 with a constant
 * a_i = gamma, Mamba2 with a data-dependent scalar) or T_i = diag(g_i) (GLA); u_i = k_i v_i^T (no beta, no erase term).
 * Row convention (state dv x dk):   S <- S diag(a_t) + v_t k_t^T,   a_t = exp(g_t)  (reading A2).
 * PAPER.md:188-200 (Table 3): T_C = (prod_t a_t) I, stored as ONE scalar, or diag(prod_t g_t), stored as the
 * dk-vector; applying it is an element-wise scaling of S.
 *
 * hypic_oracle_diag_encode: per (segment, head): E = end state from S = 0 (dv x dk) and tvec = prod_t a_t
 * ([n_seg,H] for the scalar gate, [n_seg,H,dk] for the per-channel gate), the product taken token by token.
 * A zero-length segment gives E = 0, tvec = 1.  g:[Ttot,H] or [Ttot,H,dk].
 */
int hypic_oracle_diag_encode(const float* k, const float* v, const float* g, const int32_t* cu_seqlens, int n_seg,
                             int H, int dk, int dv, int gate, double* E, double* tvec) {
  if (n_seg < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_seqlens || !E || !tvec) return 1;
  if (gate != HYPIC_ORACLE_GATE_SCALAR && gate != HYPIC_ORACLE_GATE_CHANNEL) return 1;
  const int tw = gate == HYPIC_ORACLE_GATE_CHANNEL ? dk : 1;
  const long n_units = (long)n_seg * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int s = (int)(u / H), h = (int)(u % H);
    double* Eu = E + (size_t)u * dv * dk;
    double* tu = tvec + (size_t)u * tw;
    memset(Eu, 0, sizeof(double) * (size_t)dv * dk);
    for (int c = 0; c < tw; ++c) tu[c] = 1.0;
    for (int t = cu_seqlens[s]; t < cu_seqlens[s + 1]; ++t) {
      const size_t th = (size_t)t * H + h;
      for (int c = 0; c < tw; ++c) tu[c] *= exp((double)g[th * tw + c]);
      for (int i = 0; i < dv; ++i)
        for (int c = 0; c < dk; ++c) {
          const double a = exp((double)g[th * tw + (tw == 1 ? 0 : c)]);
          Eu[(size_t)i * dk + c] = Eu[(size_t)i * dk + c] * a + (double)v[th * dv + i] * (double)k[th * dk + c];
        }
    }
  }
  return 0;
}

/*
 * hypic_oracle_diag_sequential: the same token recurrence from S_in (NULL = zeros) over each request's tokens
 * [cu_tokens[r], cu_tokens[r+1]): what composing the request's segments must reproduce (Eq. 4).
 */
int hypic_oracle_diag_sequential(const double* S_in, const float* k, const float* v, const float* g,
                                 const int32_t* cu_tokens, int R, int H, int dk, int dv, int gate, double* S_out) {
  if (R < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_tokens || !S_out) return 1;
  if (gate != HYPIC_ORACLE_GATE_SCALAR && gate != HYPIC_ORACLE_GATE_CHANNEL) return 1;
  const int tw = gate == HYPIC_ORACLE_GATE_CHANNEL ? dk : 1;
  const long n_units = (long)R * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int r = (int)(u / H), h = (int)(u % H);
    double* Su = S_out + (size_t)u * dv * dk;
    if (S_in)
      memcpy(Su, S_in + (size_t)u * dv * dk, sizeof(double) * (size_t)dv * dk);
    else
      memset(Su, 0, sizeof(double) * (size_t)dv * dk);
    for (int t = cu_tokens[r]; t < cu_tokens[r + 1]; ++t) {
      const size_t th = (size_t)t * H + h;
      for (int i = 0; i < dv; ++i)
        for (int c = 0; c < dk; ++c) {
          const double a = exp((double)g[th * tw + (tw == 1 ? 0 : c)]);
          Su[(size_t)i * dk + c] = Su[(size_t)i * dk + c] * a + (double)v[th * dv + i] * (double)k[th * dk + c];
        }
    }
  }
  return 0;
}

/*
 * hypic_oracle_diag_compose: PAPER.md:182 (Eq. 6) with the compressed transitions of Table 3: for every request and
 * head, S <- S diag(tvec_i) + E_i over the request's ordered pool ids (scalar gate: S <- tvec_i S + E_i).
 * E_pool:[P,H,dv,dk], t_pool:[P,H] or [P,H,dk], doubles.
 */
int hypic_oracle_diag_compose(const double* S_in, const double* E_pool, const double* t_pool, const int32_t* seg_ids,
                              const int32_t* cu_segs, int R, int H, int dk, int dv, int gate, double* S_out) {
  if (R < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_segs || !S_out) return 1;
  if (gate != HYPIC_ORACLE_GATE_SCALAR && gate != HYPIC_ORACLE_GATE_CHANNEL) return 1;
  const int tw = gate == HYPIC_ORACLE_GATE_CHANNEL ? dk : 1;
  const long n_units = (long)R * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int r = (int)(u / H), h = (int)(u % H);
    double* Su = S_out + (size_t)u * dv * dk;
    if (S_in)
      memcpy(Su, S_in + (size_t)u * dv * dk, sizeof(double) * (size_t)dv * dk);
    else
      memset(Su, 0, sizeof(double) * (size_t)dv * dk);
    for (int j = cu_segs[r]; j < cu_segs[r + 1]; ++j) {
      const size_t ph = (size_t)seg_ids[j] * H + h;
      const double* Ei = E_pool + ph * dv * dk;
      const double* ti = t_pool + ph * tw;
      for (int i = 0; i < dv; ++i)
        for (int c = 0; c < dk; ++c)
          Su[(size_t)i * dk + c] = Su[(size_t)i * dk + c] * ti[tw == 1 ? 0 : c] + Ei[(size_t)i * dk + c];
    }
  }
  return 0;
}

/*
 * hypic_oracle_rope_compose: state RoPE re-rotation, PAPER.md:208-214 (Eq. 7), scalar family only (T_i = t_i I commutes
 * with every rotation): "Hypic replaces each S_{C_i|0} in Equation (6) with R(p_i) S_{C_i|0}", p_i = the segment's
 * global start position.  Row convention (reading A1): the keys run along the columns of the dv x dk state,
 * so R(p) acts on every ROW of E_i as it acts on a key.  Pairing and angles (reading R1): column c < dk/2 is
 * paired with column c + dk/2, angle phi_c = p * inv_freq[c]:
 *     E'[i][c]        = E[i][c] cos(phi_c) - E[i][c + dk/2] sin(phi_c)
 *     E'[i][c + dk/2] = E[i][c] sin(phi_c) + E[i][c + dk/2] cos(phi_c)
 * then  S <- t_i S + E'_i  over the request's ordered ids.  pos:int32[cu_segs[R]] (one start position per list entry),
 * inv_freq:double[dk/2], E_pool:[P,H,dv,dk], t_pool:[P,H], doubles.  Pins: R1-R3 of tests/test_oracle_pins.py.
 */
int hypic_oracle_rope_compose(const double* S_in, const double* E_pool, const double* t_pool, const int32_t* seg_ids,
                              const int32_t* cu_segs, const int32_t* pos, const double* inv_freq, int R, int H, int dk,
                              int dv, double* S_out) {
  if (R < 0 || H <= 0 || dk <= 0 || (dk & 1) || dv <= 0 || !cu_segs || !S_out || !inv_freq) return 1;
  const int half = dk / 2;
  const long n_units = (long)R * H;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int r = (int)(u / H), h = (int)(u % H);
    double* Su = S_out + (size_t)u * dv * dk;
    if (S_in)
      memcpy(Su, S_in + (size_t)u * dv * dk, sizeof(double) * (size_t)dv * dk);
    else
      memset(Su, 0, sizeof(double) * (size_t)dv * dk);
    for (int j = cu_segs[r]; j < cu_segs[r + 1]; ++j) {
      const size_t ph = (size_t)seg_ids[j] * H + h;
      const double* Ei = E_pool + ph * dv * dk;
      const double ti = t_pool[ph];
      for (int c = 0; c < half; ++c) {
        const double phi = (double)pos[j] * inv_freq[c];
        const double cs = cos(phi), sn = sin(phi);
        for (int i = 0; i < dv; ++i) {
          const double a = Ei[(size_t)i * dk + c], b = Ei[(size_t)i * dk + c + half];
          Su[(size_t)i * dk + c] = Su[(size_t)i * dk + c] * ti + (a * cs - b * sn);
          Su[(size_t)i * dk + c + half] = Su[(size_t)i * dk + c + half] * ti + (a * sn + b * cs);
        }
      }
    }
  }
  return 0;
}

/*
 * hypic_oracle_compose: PAPER.md:182 (Eq. 6) evaluated as the chain it abbreviates (Eq. 4
 * applied once per segment), in the row convention:  S <- S T_i + E_i  for i = first .. last of the request's
 * ordered segment list.  Composition is not commutative; the order is the list order.
 * S_in:[R,H,dv,dk] doubles or NULL (zeros); pools E:[P,H,dv,dk], T:[P,H,dk,dk], float32 if pool_is_f32 else
 * float64; seg_ids:int32[cu_segs[R]] with values in [0,P); cu_segs:int32[R+1]; S_out:[R,H,dv,dk] doubles.
 * Returns 0, 1 on a bad argument, 2 on a segment id out of range.
 */
int hypic_oracle_compose(const double* S_in, const void* E_pool, const void* T_pool, int pool_is_f32,
                         const int32_t* seg_ids, const int32_t* cu_segs, int R, int P, int H, int dk, int dv,
                         double* S_out) {
  if (R < 0 || P < 0 || H <= 0 || dk <= 0 || dv <= 0 || !cu_segs || !S_out) return 1;
  for (int r = 0; r < R; ++r)
    for (int j = cu_segs[r]; j < cu_segs[r + 1]; ++j)
      if (seg_ids[j] < 0 || seg_ids[j] >= P) return 2;
  const long n_units = (long)R * H;
  const size_t se = (size_t)dv * dk, st = (size_t)dk * dk;
#pragma omp parallel for schedule(dynamic, 1)
  for (long u = 0; u < n_units; ++u) {
    const int r = (int)(u / H), h = (int)(u % H);
    double* S = S_out + (size_t)u * se;
    double* Snew = (double*)malloc(sizeof(double) * se);
    if (S_in)
      memcpy(S, S_in + (size_t)u * se, sizeof(double) * se);
    else
      memset(S, 0, sizeof(double) * se);
    for (int j = cu_segs[r]; j < cu_segs[r + 1]; ++j) {
      const size_t ph = (size_t)seg_ids[j] * H + h;
      for (int i = 0; i < dv; ++i) {
        for (int b = 0; b < dk; ++b) {
          double acc = pool_is_f32 ? (double)((const float*)E_pool)[ph * se + (size_t)i * dk + b]
                                   : ((const double*)E_pool)[ph * se + (size_t)i * dk + b];
          for (int c = 0; c < dk; ++c) {
            const double tcb = pool_is_f32 ? (double)((const float*)T_pool)[ph * st + (size_t)c * dk + b]
                                           : ((const double*)T_pool)[ph * st + (size_t)c * dk + b];
            acc += S[(size_t)i * dk + c] * tcb;
          }
          Snew[(size_t)i * dk + b] = acc;
        }
      }
      memcpy(S, Snew, sizeof(double) * se);
    }
    free(Snew);
  }
  return 0;
}
