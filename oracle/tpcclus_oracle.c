/*
 * oracle/tpcclus_oracle.c -- T1 oracle of the TPC clusterizer.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  A plain, slow, single-threaded CPU
 * restatement of what the hot path computes.  Only tests/, the smoke check
 * in __graft_entry__.py and the cpu_baseline / --impl reference legs of
 * bench.py may call it.  It shares no code, header, table or helper with
 * paper_2511_17018_b200/ (the CUDA path); the two record layouts below are
 * typed out independently from the same specification.
 *
 * What it follows.  The paper never describes the clusterizer; the
 * path is named by BASELINE.json north_star (NS) and every open detail is
 * fixed by SURVEY.md section 8(c), steps O0..O5 and readings Q1..Q23.  The
 * paper contributes the run-mode rules this oracle obeys:
 *   P:36   total order for every comparison that decides an outcome (beats())
 *   P:37-39 IEEE single precision, no FMA contraction, no fast math
 *          (build with -O2 -ffp-contract=off -fno-fast-math; SSE2 floats)
 *   P:41   "the GPU code uses only single-precision floating point" -> the
 *          finalisation O4 is float32, one rounding per operation.  The sums
 *          O3 are 32-bit integers and exact, so order of summation is moot.
 *   P:47-48 output order fixed: (sector,row,time,pad) ascending (O5).
 *
 * There is no blocking, fusion or reordering here beyond the loop nest the
 * definition states.
 *
 * Pins (tests/test_oracle_*.py): SURVEY Appendix A worked vectors
 * (tests/golden/), exact-rational correct rounding of O4, T0 (global-rank
 * brute force, oracle/t0_bruteforce.py) on exhaustive tiny maps, invariants
 * I1..I12.  Unpinned: the *choice* of conventions Q6/Q9/Q10 (thresholds,
 * suppression criterion, unit weights) -- nothing external fixes them;
 * see DESIGN.md "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* 8-byte little-endian digit record. */
typedef struct {
  uint16_t charge;
  uint16_t time;
  uint8_t pad;
  uint8_t row;
  uint8_t sector;
  uint8_t reserved;
} orc_digit;

/* 32-byte cluster record. */
typedef struct {
  float pad_mean, time_mean, sigma_pad, sigma_time;
  uint32_t q_tot;
  uint16_t q_max;
  uint16_t time_peak;
  uint8_t pad_peak, row, sector, flags;
  uint32_t reserved;
} orc_cluster;

enum { ORC_STATUS_OVERFLOW = 1u, ORC_STATUS_BAD_DIGITS = 2u };
enum { ORC_FLAG_EDGE_PAD = 1u, ORC_FLAG_EDGE_TIME = 2u, ORC_FLAG_SATURATED = 4u };

typedef struct {
  uint32_t T;          /* time bins */
  uint32_t P;          /* pads in this row */
  const uint16_t* q;   /* [T][P] */
} row_map;

/* O0 / Q8: cells outside the ranges read as 0. */
static uint32_t cell(const row_map* m, int64_t t, int64_t p) {
  if (t < 0 || p < 0 || t >= (int64_t)m->T || p >= (int64_t)m->P) return 0;
  return m->q[(size_t)t * m->P + (size_t)p];
}

/* O1 / Q7 / P:36: strict total order on cells of one (sector,row).
 * higher charge, then earlier time, then lower pad. */
static int beats(uint32_t qa, int64_t ta, int64_t pa, uint32_t qb, int64_t tb, int64_t pb) {
  if (qa != qb) return qa > qb;
  if (ta != tb) return ta < tb;
  return pa < pb;
}

/* O1: c is a peak iff q_c >= thr_peak and c beats each of its 8 neighbours. */
static int is_peak(const row_map* m, int64_t t, int64_t p, uint32_t thr_peak) {
  uint32_t qc = cell(m, t, p);
  if (qc < thr_peak) return 0;
  for (int dt = -1; dt <= 1; ++dt)
    for (int dp = -1; dp <= 1; ++dp) {
      if (dt == 0 && dp == 0) continue;
      if (!beats(qc, t, p, cell(m, t + dt, p + dp), t + dt, p + dp)) return 0;
    }
  return 1;
}

static int iabs(int x) { return x < 0 ? -x : x; }
static int imax(int a, int b) { return a > b ? a : b; }

/* O2: peak c is suppressed iff some peak c' at Chebyshev distance exactly 2
 * beats c and a common 8-neighbour m of both has q_m + noise_eps >= q_c.
 * pk is the un-updated peak set of O1. */
static int is_suppressed(const row_map* m, const uint8_t* pk, int64_t t, int64_t p,
                         uint32_t noise_eps) {
  uint32_t qc = cell(m, t, p);
  for (int dt = -2; dt <= 2; ++dt)
    for (int dp = -2; dp <= 2; ++dp) {
      if (imax(iabs(dt), iabs(dp)) != 2) continue;
      int64_t t2 = t + dt, p2 = p + dp;
      if (t2 < 0 || p2 < 0 || t2 >= (int64_t)m->T || p2 >= (int64_t)m->P) continue;
      if (!pk[(size_t)t2 * m->P + (size_t)p2]) continue;
      if (!beats(cell(m, t2, p2), t2, p2, qc, t, p)) continue;
      /* common neighbours: cells within distance 1 of both c and c' (and != either) */
      for (int mt = -1; mt <= 1; ++mt)
        for (int mp = -1; mp <= 1; ++mp) {
          if (mt == 0 && mp == 0) continue;
          int64_t tm = t + mt, pm = p + mp;
          if (imax(iabs((int)(tm - t2)), iabs((int)(pm - p2))) != 1) continue;
          if (cell(m, tm, pm) + noise_eps >= qc) return 1;
        }
    }
  return 0;
}

/* O4: float32 finalisation, every operation rounded once (RN-even), no
 * contraction.  volatile stores make the single rounding explicit even if a
 * compiler were to keep wider temporaries. */
void oracle_finalize(uint32_t Q, int32_t Sp, int32_t St, uint32_t Spp, uint32_t Stt,
                     uint32_t p_c, uint32_t t_c, float out4[4]) {
  int32_t Vp = (int32_t)(Q * Spp) - Sp * Sp; /* O3: fits, Q*Spp <= 1308161250 */
  int32_t Vt = (int32_t)(Q * Stt) - St * St;
  volatile float fQ = (float)Q;
  volatile float dp = (float)Sp / fQ;
  volatile float dt = (float)St / fQ;
  volatile float pm = (float)p_c + dp;
  volatile float tm = (float)t_c + dt;
  volatile float rp = sqrtf((float)Vp);
  volatile float rt = sqrtf((float)Vt);
  volatile float sp = rp / fQ;
  volatile float st = rt / fQ;
  out4[0] = pm;
  out4[1] = tm;
  out4[2] = sp;
  out4[3] = st;
}

/* O3 + O4 for one surviving peak.  `gated` selects reading Q10' (DESIGN.md
 * R7): a cell of the outer ring of the 5x5 window, max(|dp|,|dt|) = 2, counts only if the inner
 * cell between it and the peak -- (clamp(dt,-1,1), clamp(dp,-1,1)) -- is non-empty. */
static void make_cluster(const row_map* m, uint32_t s, uint32_t r, int64_t t, int64_t p,
                         orc_cluster* c, int gated) {
  uint32_t Q = 0, Spp = 0, Stt = 0;
  int32_t Sp = 0, St = 0;
  for (int dt = -2; dt <= 2; ++dt)
    for (int dp = -2; dp <= 2; ++dp) {
      uint32_t q = cell(m, t + dt, p + dp); /* Q8/Q10: clipped window, weight 1 */
      if (gated && (iabs(dt) == 2 || iabs(dp) == 2)) {
        int it = dt < -1 ? -1 : (dt > 1 ? 1 : dt), ip = dp < -1 ? -1 : (dp > 1 ? 1 : dp);
        if (cell(m, t + it, p + ip) == 0) q = 0; /* Q10': weight 0 */
      }
      Q += q;
      Sp += (int32_t)q * dp;
      St += (int32_t)q * dt;
      Spp += q * (uint32_t)(dp * dp);
      Stt += q * (uint32_t)(dt * dt);
    }
  float f[4];
  oracle_finalize(Q, Sp, St, Spp, Stt, (uint32_t)p, (uint32_t)t, f);
  memset(c, 0, sizeof *c);
  c->pad_mean = f[0];
  c->time_mean = f[1];
  c->sigma_pad = f[2];
  c->sigma_time = f[3];
  c->q_tot = Q;
  c->q_max = (uint16_t)cell(m, t, p);
  c->time_peak = (uint16_t)t;
  c->pad_peak = (uint8_t)p;
  c->row = (uint8_t)r;
  c->sector = (uint8_t)s;
  uint8_t fl = 0;
  if (p < 2 || p + 2 >= (int64_t)m->P) fl |= ORC_FLAG_EDGE_PAD;
  if (t < 2 || t + 2 >= (int64_t)m->T) fl |= ORC_FLAG_EDGE_TIME;
  if (c->q_max == 1023) fl |= ORC_FLAG_SATURATED;
  c->flags = fl;
  c->reserved = 0;
}

/* O3 + O4 in reading Q10'' (second half; R8): charge sharing between
 * clusters whose windows overlap.  sv = the survivor set of O2 for this row map.  The PARTNERS of a
 * survivor c are the survivors c' at Chebyshev distance exactly 2 (no two peaks are closer), i.e.
 * those whose peak cell lies on the outer ring of c's window.  A cell x of c's window that also lies
 * in the window of partners c'_1..c'_k is split with integer weights
 *     w_p(x) = (q_p >> (2 * cheb(p, x))) + 1            (peak charge, quartered per bin of distance)
 *     share_c(x) = floor(q_x * w_c(x) / (w_c(x) + sum_i w_c'_i(x)))
 * and enters the sums of O3 with that share instead of q_x.  A cell no partner reaches keeps its
 * full charge (the quotient is q_x * w / w).  A peak cell is never split: c keeps q_c in full (so
 * Q >= q_c >= 1) and takes nothing of a partner's peak cell.  Everything stays an exact integer. */
static int cheb(int64_t t1, int64_t p1, int64_t t2, int64_t p2) {
  return imax(iabs((int)(t1 - t2)), iabs((int)(p1 - p2)));
}

static void make_cluster_shared(const row_map* m, const uint8_t* sv, uint32_t s, uint32_t r, int64_t t,
                                int64_t p, orc_cluster* c) {
  uint32_t Q = 0, Spp = 0, Stt = 0;
  int32_t Sp = 0, St = 0;
  uint32_t qc = cell(m, t, p);
  for (int dt = -2; dt <= 2; ++dt)
    for (int dp = -2; dp <= 2; ++dp) {
      int64_t tx = t + dt, px = p + dp;
      uint32_t q = cell(m, tx, px); /* Q8: clipped window */
      if (q == 0) continue;
      uint32_t wc = (qc >> (2 * cheb(t, p, tx, px))) + 1, den = wc;
      int partner_peak = 0;
      for (int et = -2; et <= 2; ++et)       /* the partners: survivors on the outer ring of c */
        for (int ep = -2; ep <= 2; ++ep) {
          if (imax(iabs(et), iabs(ep)) != 2) continue;
          int64_t t2 = t + et, p2 = p + ep;
          if (t2 < 0 || p2 < 0 || t2 >= (int64_t)m->T || p2 >= (int64_t)m->P) continue;
          if (!sv[(size_t)t2 * m->P + (size_t)p2]) continue;
          int d2 = cheb(t2, p2, tx, px);
          if (d2 > 2) continue;                /* x is outside that partner's window */
          if (d2 == 0) partner_peak = 1;       /* x is that partner's own peak cell */
          den += (cell(m, t2, p2) >> (2 * d2)) + 1;
        }
      uint32_t share = q * wc / den;
      if (dt == 0 && dp == 0) share = q;       /* the peak cell is c's alone ... */
      if (partner_peak) share = 0;             /* ... and a partner's peak cell is the partner's */
      Q += share;
      Sp += (int32_t)share * dp;
      St += (int32_t)share * dt;
      Spp += share * (uint32_t)(dp * dp);
      Stt += share * (uint32_t)(dt * dt);
    }
  float f[4];
  oracle_finalize(Q, Sp, St, Spp, Stt, (uint32_t)p, (uint32_t)t, f);
  memset(c, 0, sizeof *c);
  c->pad_mean = f[0];
  c->time_mean = f[1];
  c->sigma_pad = f[2];
  c->sigma_time = f[3];
  c->q_tot = Q;
  c->q_max = (uint16_t)qc;
  c->time_peak = (uint16_t)t;
  c->pad_peak = (uint8_t)p;
  c->row = (uint8_t)r;
  c->sector = (uint8_t)s;
  uint8_t fl = 0;
  if (p < 2 || p + 2 >= (int64_t)m->P) fl |= ORC_FLAG_EDGE_PAD;
  if (t < 2 || t + 2 >= (int64_t)m->T) fl |= ORC_FLAG_EDGE_TIME;
  if (c->q_max == 1023) fl |= ORC_FLAG_SATURATED;
  c->flags = fl;
  c->reserved = 0;
}

/*
 * Whole path O0..O5.  Returns the true number of clusters (also when it
 * exceeds `capacity`; then ORC_STATUS_OVERFLOW is set and only the first
 * `capacity` clusters in output order are stored), or -1 on allocation failure.
 * If dbg_map != NULL it must hold n_sectors * sum_r(T*n_pads[r]) uint16 and
 * receives the O0 map in [sector][row][time][pad] order (for map-level pins).
 */
int64_t oracle_clusterize_ex(uint32_t n_sectors, uint32_t n_rows, uint32_t n_time,
                             const uint16_t* n_pads, uint32_t thr_peak, uint32_t noise_eps,
                             const orc_digit* digits, uint64_t n_digits, orc_cluster* out,
                             uint64_t capacity, uint32_t* status, uint16_t* dbg_map, int cog_gated);

int64_t oracle_clusterize(uint32_t n_sectors, uint32_t n_rows, uint32_t n_time,
                          const uint16_t* n_pads, uint32_t thr_peak, uint32_t noise_eps,
                          const orc_digit* digits, uint64_t n_digits, orc_cluster* out,
                          uint64_t capacity, uint32_t* status, uint16_t* dbg_map) {
  return oracle_clusterize_ex(n_sectors, n_rows, n_time, n_pads, thr_peak, noise_eps, digits, n_digits, out,
                              capacity, status, dbg_map, 0);
}

int64_t oracle_clusterize_ex(uint32_t n_sectors, uint32_t n_rows, uint32_t n_time,
                             const uint16_t* n_pads, uint32_t thr_peak, uint32_t noise_eps,
                             const orc_digit* digits, uint64_t n_digits, orc_cluster* out,
                             uint64_t capacity, uint32_t* status, uint16_t* dbg_map, int cog_gated) {
  uint32_t st = 0;
  uint64_t n_out = 0;

  /* per-row offsets inside one sector's map */
  size_t* row_off = (size_t*)malloc(((size_t)n_rows + 1) * sizeof(size_t));
  if (!row_off) return -1;
  row_off[0] = 0;
  for (uint32_t r = 0; r < n_rows; ++r)
    row_off[r + 1] = row_off[r] + (size_t)n_time * n_pads[r];
  size_t sector_cells = row_off[n_rows];

  /* bucket digit indices by sector (bookkeeping only; O0's validity rule Q4
   * for the sector field is applied here, the rest below) */
  uint64_t* first = (uint64_t*)calloc((size_t)n_sectors + 1, sizeof(uint64_t));
  uint64_t* order = (uint64_t*)malloc((n_digits ? n_digits : 1) * sizeof(uint64_t));
  uint64_t* fill = (uint64_t*)calloc((size_t)n_sectors + 1, sizeof(uint64_t));
  uint16_t* q = (uint16_t*)malloc((sector_cells ? sector_cells : 1) * sizeof(uint16_t));
  uint8_t* pk = (uint8_t*)malloc(sector_cells ? sector_cells : 1);
  uint8_t* sv = (uint8_t*)malloc(sector_cells ? sector_cells : 1);
  if (!first || !order || !fill || !q || !pk || !sv) {
    free(row_off); free(first); free(order); free(fill); free(q); free(pk); free(sv);
    return -1;
  }
  for (uint64_t i = 0; i < n_digits; ++i) {
    if (digits[i].sector >= n_sectors) { st |= ORC_STATUS_BAD_DIGITS; continue; }
    first[digits[i].sector + 1]++;
  }
  for (uint32_t s = 0; s < n_sectors; ++s) first[s + 1] += first[s];
  for (uint64_t i = 0; i < n_digits; ++i) {
    if (digits[i].sector >= n_sectors) continue;
    uint32_t s = digits[i].sector;
    order[first[s] + fill[s]++] = i;
  }

  for (uint32_t s = 0; s < n_sectors; ++s) {
    /* O0: map = 0, then max-merge every valid digit */
    memset(q, 0, sector_cells * sizeof(uint16_t));
    for (uint64_t k = first[s]; k < first[s + 1]; ++k) {
      const orc_digit* d = &digits[order[k]];
      if (d->row >= n_rows || d->pad >= n_pads[d->row] || d->time >= n_time) {
        st |= ORC_STATUS_BAD_DIGITS;   /* Q4: ignore + flag */
        continue;
      }
      uint16_t qq = d->charge > 1023 ? 1023 : d->charge; /* Q4: clamp */
      if (qq == 0) continue;                              /* Q4: ignore */
      uint16_t* c = &q[row_off[d->row] + (size_t)d->time * n_pads[d->row] + d->pad];
      if (qq > *c) *c = qq;                               /* Q5: maximum wins */
    }
    if (dbg_map) memcpy(dbg_map + (size_t)s * sector_cells, q, sector_cells * sizeof(uint16_t));

    for (uint32_t r = 0; r < n_rows; ++r) {
      row_map m = { n_time, n_pads[r], q + row_off[r] };
      uint8_t* pkr = pk + row_off[r];
      /* O1: peak set */
      for (uint32_t t = 0; t < n_time; ++t)
        for (uint32_t p = 0; p < m.P; ++p)
          pkr[(size_t)t * m.P + p] = (uint8_t)is_peak(&m, t, p, thr_peak);
      /* O2: survivor set (against the un-updated peak set) */
      uint8_t* svr = sv + row_off[r];
      for (uint32_t t = 0; t < n_time; ++t)
        for (uint32_t p = 0; p < m.P; ++p)
          svr[(size_t)t * m.P + p] = (uint8_t)(pkr[(size_t)t * m.P + p] && !is_suppressed(&m, pkr, t, p, noise_eps));
      /* O3 + O4 + O5: survivors in (time,pad) order; cog_gated: 0 = Q10, 1 = Q10', 2 = Q10'' */
      for (uint32_t t = 0; t < n_time; ++t)
        for (uint32_t p = 0; p < m.P; ++p) {
          if (!svr[(size_t)t * m.P + p]) continue;
          if (n_out < capacity) {
            if (cog_gated == 2) make_cluster_shared(&m, svr, s, r, t, p, &out[n_out]);
            else make_cluster(&m, s, r, t, p, &out[n_out], cog_gated);
          } else st |= ORC_STATUS_OVERFLOW;
          ++n_out;
        }
    }
  }
  free(row_off); free(first); free(order); free(fill); free(q); free(pk); free(sv);
  if (status) *status = st;
  return (int64_t)n_out;
}

/* Step-level entry for pins: O1 (+ optionally O2) flags of a single row map.
 * flags_out[t*P+p]: bit0 = peak after O1, bit1 = survives O2. */
void oracle_row_flags(uint32_t T, uint32_t P, const uint16_t* q, uint32_t thr_peak,
                      uint32_t noise_eps, uint8_t* flags_out) {
  row_map m = { T, P, q };
  uint8_t* pk = (uint8_t*)malloc((size_t)T * P ? (size_t)T * P : 1);
  for (uint32_t t = 0; t < T; ++t)
    for (uint32_t p = 0; p < P; ++p) pk[(size_t)t * P + p] = (uint8_t)is_peak(&m, t, p, thr_peak);
  for (uint32_t t = 0; t < T; ++t)
    for (uint32_t p = 0; p < P; ++p) {
      uint8_t f = pk[(size_t)t * P + p];
      if (f && !is_suppressed(&m, pk, t, p, noise_eps)) f |= 2;
      flags_out[(size_t)t * P + p] = f;
    }
  free(pk);
}

uint32_t oracle_sizeof_digit(void) { return (uint32_t)sizeof(orc_digit); }
uint32_t oracle_sizeof_cluster(void) { return (uint32_t)sizeof(orc_cluster); }
