/*
 * oracle/ic_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, step-by-step C implementation of the charge-conserving
 * Metropolis algorithm with "coupled pairs" of arXiv:2301.11735 (Budrin et al.),
 * written from the paper and from the readings listed
 * in DESIGN.md ("Readings of the paper").  It is the authority the CUDA library
 * (paper_2301_11735_b200/csrc) is compared against, bit for bit.
 *
 * Rules (see the task statement, section 3):
 *   - only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference legs may load this file;
 *   - it shares no code, header, table or constant generator with the CUDA
 *     path; the CUDA path never calls into it;
 *   - fp64 everywhere floating point is used, no FMA contraction
 *     (compile with -ffp-contract=off), integers for all lattice work.
 *
 * Notation follows the paper: site state S = +-1 (charge) or s = +-1/2 with
 * S = 0 (magnetic), sigma = 2(1-S^2)s in {+1,-1,0}  (sec. 2.1).
 * Public site code c: 0 -> sigma=+1, 1 -> sigma=-1, 2 -> S=+1, 3 -> S=-1.
 * Energy, eq. (3):
 *      E = Delta*n2 + V*bV + (J/4)*bJ,
 *      n2 = sum_i S_i^2, bV = sum_<ij> S_i S_j, bJ = sum_<ij> sigma_i sigma_j,
 * each site contributing its +x and +y bond, periodic.
 * Constraint, eq. (2): sum_i S_i = Q = const.
 *
 * Parity pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
 *   philox4x32      10 rounds: known-answer vectors of Salmon et al. (tests/golden/philox_kat.txt); 7 rounds (the
 *                   update stream): the same vectors with the last three rounds inverted in the test
 *   pair_update     dE closed form (eq. 4,5 with the corrected E_J) == direct
 *                   energy difference from eq. (3) (asserted on EVERY move here,
 *                   and against orc_recompute in the tests); sum S conserved
 *   proposal table  class sizes 1/4/6, charge kept, uniform
 *                   sampling of the fixed-Q space at Delta=V=J=0 (closed form)
 *   schedules S0,S1 exact canonical <E>,<E^2>,<M^2> from brute-force enumeration
 *                   (oracle/ic_enum.c) on 3x3, 2x4, 4x4 within 3 standard errors;
 *                   S1 structure: exact cover, conflict-freeness, order independence
 *   threshold       closed form against math.exp, monotonicity, limits
 *   orc_recompute   brute-force Python loops on tiny lattices, frozen lattice n=+-1
 *   init (U0)       exact counts; "parity unpinned" by the paper (recipe is ours)
 *   chi, sweep unit "parity unpinned" by the paper (readings G8, G9);
 *                   <M^2> itself is pinned by enumeration
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "ic_oracle.h"

/* S(c) and sigma(c) for the public site code. */
static const int S_OF[4] = {0, 0, +1, -1};
static const int SG_OF[4] = {+1, -1, 0, 0};

/* ------------------------------------------------------------------------- */
/* U3: Philox4x32-R (Salmon, Moraes, Dror, Shaw, SC'11) from its definition.  */
/* DESIGN.md reading G5: the paper only says "randomly selected" */
/* ------------------------------------------------------------------------- */
void orc_philox4x32(const uint32_t ctr[4], const uint32_t key[2], int rounds, uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < rounds; ++round) {
    uint64_t p0 = M0 * (uint64_t)c0;
    uint64_t p1 = M1 * (uint64_t)c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  orc_philox4x32(ctr, key, 10, out);
}

/* Counter layout:
 *   ctr = (c0, c1, c2, replica | tag<<28),   key = (seed lo, seed hi)          */
/* tags 0..3 here; oracle/ic_variants.c uses 4..7 */
enum { TAG_UPDATE = 0, TAG_SCHED = 1, TAG_INIT = 2, TAG_S0 = 3 };

/* Rounds of the update stream: ORC_UPDATE_ROUNDS (7, what the library is built with) unless a test asks for another
 * member of the family -- tests/test_oracle_pins.py compares the sampled <E> and C at 7 and at 10 rounds.  Set between
 * runs only (the sweeps read it from several threads). */
static int g_update_rounds = ORC_UPDATE_ROUNDS;
int orc_set_update_rounds(int rounds) {
  if (rounds < 1 || rounds > 16) return -1;
  g_update_rounds = rounds;
  return 0;
}
int orc_get_update_rounds(void) { return g_update_rounds; }

void orc_philox_tagged(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2,
                       uint32_t replica, uint32_t tag, uint32_t out[4]) {
  uint32_t ctr[4] = {c0, c1, c2, (replica & 0x0FFFFFFFu) | (tag << 28)};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  /* DESIGN.md G5: the update stream of schedule S1 (one block per four pair updates) is Philox4x32-7, the
   * seven-round member of the family (Salmon et al. report 7 rounds as the fewest that pass BigCrush, 10 as the
   * default with a safety margin); every other stream (schedule, stage 1, S0 and the variants) uses 10 rounds. */
  orc_philox4x32(ctr, key, tag == TAG_UPDATE ? g_update_rounds : 10, out);
}

/* ------------------------------------------------------------------------- */
/* U2: acceptance threshold.  Metropolis min(1, exp(-dE/T)) as a  */
/* 29-bit integer: the move is accepted iff (w >> 3) < t29  (G10).   */
/* ------------------------------------------------------------------------- */
uint32_t orc_threshold(double delta, double V, double J, int dn2, int dV, int dJ, double T) {
  double dE = (delta * (double)dn2 + V * (double)dV) + (0.25 * J) * (double)dJ;
  if (dE <= 0.0) return 536870912u; /* 2^29: always accepted */
  double p = exp(-dE / T);
  double t = floor(p * 536870912.0);
  if (t < 1.0) t = 1.0;                 /* never exactly zero (resolution 2^-29) */
  if (t > 536870911.0) t = 536870911.0; /* strictly below "always"               */
  return (uint32_t)t;
}

/* ------------------------------------------------------------------------- */
/* Lattice helpers                                                            */
/* ------------------------------------------------------------------------- */
static inline int64_t site(const orc_state* st, int x, int y) {
  int Lx = st->Lx, Ly = st->Ly;
  x %= Lx; if (x < 0) x += Lx;
  y %= Ly; if (y < 0) y += Ly;
  return (int64_t)y * Lx + x;
}

/* Full recomputation of (n2, bV, bJ, M, Ms, Q) from eq. (3): every site
 * contributes its +x and +y bond (a dimension of size 2 gives a double bond). */
void orc_recompute(const int8_t* code, int Lx, int Ly, int64_t out6[6]) {
  int64_t n2 = 0, bV = 0, bJ = 0, M = 0, Ms = 0, Q = 0;
  for (int y = 0; y < Ly; ++y) {
    for (int x = 0; x < Lx; ++x) {
      int c = code[(int64_t)y * Lx + x];
      int cr = code[(int64_t)y * Lx + (x + 1) % Lx];
      int cd = code[(int64_t)((y + 1) % Ly) * Lx + x];
      n2 += S_OF[c] * S_OF[c];
      bV += S_OF[c] * S_OF[cr] + S_OF[c] * S_OF[cd];
      bJ += SG_OF[c] * SG_OF[cr] + SG_OF[c] * SG_OF[cd];
      M += SG_OF[c];
      Ms += (((x + y) & 1) ? -1 : +1) * SG_OF[c];
      Q += S_OF[c];
    }
  }
  out6[0] = n2; out6[1] = bV; out6[2] = bJ; out6[3] = M; out6[4] = Ms; out6[5] = Q;
}

/* Energy of all bonds that touch site a or site b, plus their on-site terms,
 * straight from eq. (3).  A bond is identified by (site, direction): the +x or
 * +y bond of that site.  The bonds touching a site i are (i,+x), (i,+y),
 * (i-x,+x), (i-y,+y); duplicates between a's and b's lists are skipped.       */
static void local_energy(const orc_state* st, const int8_t* code, int xa, int ya, int xb, int yb,
                         int64_t* n2, int64_t* bV, int64_t* bJ) {
  int64_t bs[8]; int bd[8]; int nb = 0;
  const int px[2] = {xa, xb}, py[2] = {ya, yb};
  for (int k = 0; k < 2; ++k) {
    int64_t cand_s[4]; int cand_d[4];
    cand_s[0] = site(st, px[k], py[k]);     cand_d[0] = 0; /* (i,+x)   */
    cand_s[1] = site(st, px[k], py[k]);     cand_d[1] = 1; /* (i,+y)   */
    cand_s[2] = site(st, px[k] - 1, py[k]); cand_d[2] = 0; /* (i-x,+x) */
    cand_s[3] = site(st, px[k], py[k] - 1); cand_d[3] = 1; /* (i-y,+y) */
    for (int c = 0; c < 4; ++c) {
      int dup = 0;
      for (int j = 0; j < nb; ++j) if (bs[j] == cand_s[c] && bd[j] == cand_d[c]) dup = 1;
      if (!dup) { bs[nb] = cand_s[c]; bd[nb] = cand_d[c]; ++nb; }
    }
  }
  int64_t v = 0, j4 = 0;
  for (int j = 0; j < nb; ++j) {
    int x = (int)(bs[j] % st->Lx), y = (int)(bs[j] / st->Lx);
    int64_t other = bd[j] == 0 ? site(st, x + 1, y) : site(st, x, y + 1);
    int c0 = code[bs[j]], c1 = code[other];
    v += S_OF[c0] * S_OF[c1];
    j4 += SG_OF[c0] * SG_OF[c1];
  }
  int ca = code[site(st, xa, ya)], cb = code[site(st, xb, yb)];
  *n2 = S_OF[ca] * S_OF[ca] + S_OF[cb] * S_OF[cb];
  *bV = v; *bJ = j4;
}

/* ------------------------------------------------------------------------- */
/* U1: one coupled-pair update (sec. 3.1).                     */
/* The table of two-site configurations per pair charge q in the paper's       */
/* listing order: 1 / 4 / 6 configurations.                      */
/* ------------------------------------------------------------------------- */
enum { C_SP = 0, C_SM = 1, C_CP = 2, C_CM = 3 }; /* sigma+, sigma-, S=+1, S=-1 */
static const int8_t PAIR_TABLE_Q1P[4][2] = {{C_CP, C_SP}, {C_CP, C_SM}, {C_SP, C_CP}, {C_SM, C_CP}};
static const int8_t PAIR_TABLE_Q1M[4][2] = {{C_CM, C_SP}, {C_CM, C_SM}, {C_SP, C_CM}, {C_SM, C_CM}};
static const int8_t PAIR_TABLE_Q0[6][2] = {{C_CP, C_CM}, {C_CM, C_CP}, {C_SP, C_SP},
                                            {C_SM, C_SM}, {C_SP, C_SM}, {C_SM, C_SP}};

int orc_pair_table(int q, int idx, int8_t out2[2]) {
  if (q == 2) { if (idx != 0) return 0; out2[0] = C_CP; out2[1] = C_CP; return 1; }
  if (q == -2) { if (idx != 0) return 0; out2[0] = C_CM; out2[1] = C_CM; return 1; }
  if (q == 1) { if (idx < 0 || idx >= 4) return 0; out2[0] = PAIR_TABLE_Q1P[idx][0]; out2[1] = PAIR_TABLE_Q1P[idx][1]; return 1; }
  if (q == -1) { if (idx < 0 || idx >= 4) return 0; out2[0] = PAIR_TABLE_Q1M[idx][0]; out2[1] = PAIR_TABLE_Q1M[idx][1]; return 1; }
  if (q == 0) { if (idx < 0 || idx >= 6) return 0; out2[0] = PAIR_TABLE_Q0[idx][0]; out2[1] = PAIR_TABLE_Q0[idx][1]; return 1; }
  return 0;
}

static void die(const char* msg) {
  fprintf(stderr, "ic_oracle: internal check failed: %s\n", msg);
  abort();
}

/* One attempted move of the coupled pair a=(xa,ya), b=(xb,yb) with the 32-bit
 * random word w:  proposal index r = w & 7, acceptance by (w >> 3) < t29.
 * Returns 1 if the lattice changed.                                           */
int orc_pair_update(orc_state* st, int8_t* code, int xa, int ya, int xb, int yb, uint32_t w, double T) {
  int64_t ia = site(st, xa, ya), ib = site(st, xb, yb);
  if (ia == ib) die("pair with a == b");
  st->n_attempt++;
  /* 1. charge of the pair (q = S_a + S_b, reading G2) */
  int ca = code[ia], cb = code[ib];
  int q = S_OF[ca] + S_OF[cb];
  /* 2. q = +-2: nothing to do */
  if (q == 2 || q == -2) { st->n_null++; return 0; }
  /* 3. draw the new two-site configuration with the same q.
   *    r = 3 low bits of w; |q|=1: 4 candidates, index r&3; q=0: 6 candidates,
   *    r in 0..5, r = 6,7 proposes nothing (reading G3: exact uniformity, the
   *    current configuration is one of the candidates).                        */
  int r = (int)(w & 7u);
  int8_t nw[2];
  if (q == 0) {
    if (r >= 6) { st->n_null++; return 0; }
    orc_pair_table(0, r, nw);
  } else {
    orc_pair_table(q, r & 3, nw);
  }
  int na = nw[0], nb = nw[1];
  if (S_OF[na] + S_OF[nb] != q) die("proposal changes the pair charge");
  /* 4. null move */
  if (na == ca && nb == cb) { st->n_null++; return 0; }
  /* 5. neighbour sums over the 4 slots of a and of b, current lattice; adj =
   *    number of a's slots that are b ("the sum over <a> includes
   *    S_b0")                                                                   */
  const int dx[4] = {+1, -1, 0, 0}, dy[4] = {0, 0, +1, -1};
  int nSa = 0, nGa = 0, nSb = 0, nGb = 0, adj = 0;
  for (int k = 0; k < 4; ++k) {
    int64_t ja = site(st, xa + dx[k], ya + dy[k]);
    int64_t jb = site(st, xb + dx[k], yb + dy[k]);
    nSa += S_OF[(int)code[ja]]; nGa += SG_OF[(int)code[ja]];
    nSb += S_OF[(int)code[jb]]; nGb += SG_OF[(int)code[jb]];
    if (ja == ib) ++adj;
  }
  /* 6. energy change: eq. (4) distant / eq. (5) neighbouring sites, with the
   *    corrected spin term (reading G1):
   *      E_Delta = S_a1^2 + S_b1^2 - S_a0^2 - S_b0^2
   *      E_V     = dS_a nS_a + dS_b nS_b + adj dS_a dS_b      (dS_b = -dS_a)
   *      E_J     = dsig_a nsig_a + dsig_b nsig_b + adj dsig_a dsig_b          */
  int dSa = S_OF[na] - S_OF[ca], dSb = S_OF[nb] - S_OF[cb];
  int dGa = SG_OF[na] - SG_OF[ca], dGb = SG_OF[nb] - SG_OF[cb];
  if (dSa + dSb != 0) die("dS_a + dS_b != 0");
  int dn2 = S_OF[na] * S_OF[na] + S_OF[nb] * S_OF[nb] - S_OF[ca] * S_OF[ca] - S_OF[cb] * S_OF[cb];
  int dV = dSa * nSa + dSb * nSb + adj * dSa * dSb;
  int dJ = dGa * nGa + dGb * nGb + adj * dGa * dGb;
  /*    authority: E(new) - E(old) over the touched bonds, straight from eq. (3) */
  {
    int64_t o2, oV, oJ, m2, mV, mJ;
    local_energy(st, code, xa, ya, xb, yb, &o2, &oV, &oJ);
    code[ia] = (int8_t)na; code[ib] = (int8_t)nb;
    local_energy(st, code, xa, ya, xb, yb, &m2, &mV, &mJ);
    code[ia] = (int8_t)ca; code[ib] = (int8_t)cb;
    if (m2 - o2 != dn2 || mV - oV != dV || mJ - oJ != dJ) die("closed-form dE != direct dE");
  }
  /* 7. Metropolis acceptance, integer form (U2) */
  uint32_t t29 = orc_threshold(st->delta, st->V, st->J, dn2, dV, dJ, T);
  if (!((w >> 3) < t29)) return 0;
  /* 8. accept */
  code[ia] = (int8_t)na; code[ib] = (int8_t)nb;
  st->n2 += dn2; st->bV += dV; st->bJ += dJ;
  st->M += dGa + dGb;
  st->Ms += (((xa + ya) & 1) ? -1 : +1) * dGa + (((xb + yb) & 1) ? -1 : +1) * dGb;
  st->n_accept++;
  return 1;
}

/* ------------------------------------------------------------------------- */
/* U0: stage 1: a configuration with the prescribed charge.   */
/* All sites magnetic with random sigma, then nplus sites S=+1 and nminus      */
/* sites S=-1 at distinct random sites (selection sampling, exact counts).     */
/* ------------------------------------------------------------------------- */
void orc_init_state(int8_t* code, int Lx, int Ly, int64_t nplus, int64_t nminus, uint64_t seed, int replica) {
  int64_t N = (int64_t)Lx * Ly, K = nplus + nminus, picked = 0, plus = 0;
  for (int64_t i = 0; i < N; ++i) {
    uint32_t w[4];
    orc_philox_tagged(seed, (uint32_t)(i & 0xFFFFFFFF), (uint32_t)(i >> 32), 0, (uint32_t)replica, TAG_INIT, w);
    int c = (w[0] & 1u) ? C_SM : C_SP;
    if ((int64_t)(((uint64_t)w[1] * (uint64_t)(N - i)) >> 32) < (K - picked)) {
      if ((int64_t)(((uint64_t)w[2] * (uint64_t)(K - picked)) >> 32) < (nplus - plus)) { c = C_CP; ++plus; }
      else c = C_CM;
      ++picked;
    }
    code[i] = (int8_t)c;
  }
}

void orc_attach(orc_state* st, const int8_t* code) {
  int64_t o[6];
  orc_recompute(code, st->Lx, st->Ly, o);
  st->n2 = o[0]; st->bV = o[1]; st->bJ = o[2]; st->M = o[3]; st->Ms = o[4]; st->Q = o[5];
}

/* ------------------------------------------------------------------------- */
/* U5: measurement after a sweep                              */
/* ------------------------------------------------------------------------- */
void orc_measure(orc_state* st, int64_t* trace_row) {
  double E = (st->delta * (double)st->n2 + st->V * (double)st->bV) + (0.25 * st->J) * (double)st->bJ;
  double M = (double)st->M, Ms = (double)st->Ms;
  st->sumE += E; st->sumE2 += E * E;
  st->sumM += M; st->sumM2 += M * M; st->sumAbsM += fabs(M);
  st->sumMs += Ms; st->sumMs2 += Ms * Ms; st->sumAbsMs += fabs(Ms);
  st->nmeas += 1;
  if (trace_row) {
    trace_row[0] = st->n2; trace_row[1] = st->bV; trace_row[2] = st->bJ;
    trace_row[3] = st->M; trace_row[4] = st->Ms; trace_row[5] = st->Q;
  }
}

void orc_reset_observables(orc_state* st) {
  st->nmeas = 0;
  st->sumE = st->sumE2 = st->sumM = st->sumM2 = st->sumAbsM = 0.0;
  st->sumMs = st->sumMs2 = st->sumAbsMs = 0.0;
}

/* ------------------------------------------------------------------------- */
/* U4: schedules                                                              */
/* ------------------------------------------------------------------------- */

/* S1 parameters of sweep s: words z = Philox(ctr=(0,0,s,TAG_SCHED)), the same
 * for all replicas (precedent: identical maps for all copies).
 *   even s -> FAR sweep:  mx = 2*(z0 & (L/2-1))+1, my = 2*(z1 & (L/2-1))+1
 *   odd  s -> NEAR sweep: o = z0 & 1 (0 horizontal, 1 vertical), off = z1 & 3 */
void orc_schedule_params(int L, uint64_t seed, uint64_t sweep, int32_t out4[4]) {
  uint32_t z[4];
  orc_philox_tagged(seed, 0, 0, (uint32_t)sweep, 0, TAG_SCHED, z);
  if ((sweep & 1) == 0) {
    out4[0] = 0;
    out4[1] = (int32_t)(2 * (z[0] & (uint32_t)(L / 2 - 1)) + 1);
    out4[2] = (int32_t)(2 * (z[1] & (uint32_t)(L / 2 - 1)) + 1);
    out4[3] = 0;
  } else {
    out4[0] = 1;
    out4[1] = (int32_t)(z[0] & 1u);
    out4[2] = (int32_t)(z[1] & 3u);
    out4[3] = 0;
  }
}

/* Random-number address of the pair whose slot site is (x, y) (the a-site; the b-site for horizontal dominoes):
 * Philox block counter c0 = 4*(X >> 2) + (x & 3) with X = x >> 2, c1 = y, and the word X & 3 of the block, so that
 * four consecutive sites x, x+4, x+8, x+12 of one row share a block (U3).                                */
static void rng_address(int x, int y, uint32_t* c0, uint32_t* c1, uint32_t* word) {
  int X = x >> 2;
  *c0 = (uint32_t)(((X >> 2) << 2) | (x & 3)); *c1 = (uint32_t)y; *word = (uint32_t)(X & 3);
}

/* The k-th candidate a-site of phase `phase` of sweep-type `par`: returns 1 and
 * fills the pair and its random-number address (c0, c1, word) if (x, y) is an
 * a-site.  Pairs of a phase are enumerated by ascending y, then ascending x.   */
static int s1_pair_at(int L, const int32_t par[4], int phase, int x, int y,
                      int* xb, int* yb, uint32_t* c0, uint32_t* c1, uint32_t* word) {
  if (par[0] == 0) { /* FAR: colour `phase`, a-sites have even x, b = (x^mx, y^my) */
    int mx = par[1], my = par[2];
    if (((x + y) & 1) != phase || (x & 1)) return 0;
    *xb = x ^ mx; *yb = y ^ my;
    rng_address(x, y, c0, c1, word);
    return 1;
  }
  int o = par[1], off = par[2];
  if (o == 0) { /* horizontal dominoes: u = x, v = y */
    if (((x - off - 2 * ((y + phase) & 1)) & 3) != 0) return 0;
    *xb = (x + 1) % L; *yb = y;
    rng_address(*xb, y, c0, c1, word); /* addressed by the b-site */
    return 1;
  }
  /* vertical dominoes: u = y, v = x */
  if (((y - off - 2 * ((x + phase) & 1)) & 3) != 0) return 0;
  *xb = x; *yb = (y + 1) % L;
  rng_address(x, y, c0, c1, word);
  return 1;
}

/* pairs(sweep, phase) as explicit lists (tests only; small L). Returns count. */
int64_t orc_schedule_s1(int L, uint64_t seed, uint64_t sweep, int phase,
                        int64_t* ia, int64_t* ib, uint32_t* c0, uint32_t* c1, uint32_t* word) {
  int32_t par[4];
  orc_schedule_params(L, seed, sweep, par);
  int64_t n = 0;
  for (int y = 0; y < L; ++y)
    for (int x = 0; x < L; ++x) {
      int xb, yb; uint32_t a0, a1, aw;
      if (!s1_pair_at(L, par, phase, x, y, &xb, &yb, &a0, &a1, &aw)) continue;
      ia[n] = (int64_t)y * L + x; ib[n] = (int64_t)yb * L + xb;
      c0[n] = a0; c1[n] = a1; word[n] = aw; ++n;
    }
  return n;
}

static int is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

/* S1 "colour/XOR + brick" production schedule.  order: 0 ascending,
 * 1 descending (the result must not depend on it: validity condition V2).
 * trace: NULL or [nsweeps][6] (n2,bV,bJ,M,Ms,Q after each sweep).             */
int orc_sweep_s1(orc_state* st, int8_t* code, double T, int64_t nsweeps, int order, int64_t* trace) {
  int L = st->Lx;
  if (st->Lx != st->Ly || !is_pow2(L) || L < 4) return -1;
  if (!(T > 0.0)) return -2;
  for (int64_t s = 0; s < nsweeps; ++s) {
    int32_t par[4];
    orc_schedule_params(L, st->seed, st->sweep, par);
    for (int phase = 0; phase < 2; ++phase) {
      for (int yy = 0; yy < L; ++yy) {
        int y = order ? L - 1 - yy : yy;
        for (int xx = 0; xx < L; ++xx) {
          int x = order ? L - 1 - xx : xx;
          int xb, yb; uint32_t c0, c1, word, w[4];
          if (!s1_pair_at(L, par, phase, x, y, &xb, &yb, &c0, &c1, &word)) continue;
          orc_philox_tagged(st->seed, c0, c1, (uint32_t)(2 * st->sweep + (uint64_t)phase),
                        (uint32_t)st->replica, TAG_UPDATE, w);
          orc_pair_update(st, code, x, y, xb, yb, w[word], T);
        }
      }
    }
    orc_measure(st, trace ? trace + 6 * s : NULL);
    st->sweep += 1;
  }
  return 0;
}

/* The same S1 sweep with the rows of a phase spread over OpenMP threads.  By
 * validity condition V2 (no site of one pair equals or neighbours a site of
 * another pair of the same phase) the result is identical to orc_sweep_s1; the
 * tests check that.  Used to keep full-size parity runs and the timed CPU
 * baseline short.  Each thread accumulates into a private copy of the state.  */
int orc_sweep_s1_mt(orc_state* st, int8_t* code, double T, int64_t nsweeps, int nthreads, int64_t* trace) {
  int L = st->Lx;
  if (st->Lx != st->Ly || !is_pow2(L) || L < 4) return -1;
  if (!(T > 0.0)) return -2;
  if (nthreads < 1) nthreads = 1;
  for (int64_t s = 0; s < nsweeps; ++s) {
    int32_t par[4];
    orc_schedule_params(L, st->seed, st->sweep, par);
    for (int phase = 0; phase < 2; ++phase) {
      int64_t d_n2 = 0, d_bV = 0, d_bJ = 0, d_M = 0, d_Ms = 0, d_att = 0, d_acc = 0, d_null = 0;
#pragma omp parallel for schedule(static) num_threads(nthreads) \
    reduction(+ : d_n2, d_bV, d_bJ, d_M, d_Ms, d_att, d_acc, d_null)
      for (int y = 0; y < L; ++y) {
        orc_state loc = *st;
        loc.n2 = loc.bV = loc.bJ = loc.M = loc.Ms = 0;
        loc.n_attempt = loc.n_accept = loc.n_null = 0;
        for (int x = 0; x < L; ++x) {
          int xb, yb; uint32_t c0, c1, word, w[4];
          if (!s1_pair_at(L, par, phase, x, y, &xb, &yb, &c0, &c1, &word)) continue;
          orc_philox_tagged(st->seed, c0, c1, (uint32_t)(2 * st->sweep + (uint64_t)phase),
                        (uint32_t)st->replica, TAG_UPDATE, w);
          orc_pair_update(&loc, code, x, y, xb, yb, w[word], T);
        }
        d_n2 += loc.n2; d_bV += loc.bV; d_bJ += loc.bJ; d_M += loc.M; d_Ms += loc.Ms;
        d_att += loc.n_attempt; d_acc += loc.n_accept; d_null += loc.n_null;
      }
      st->n2 += d_n2; st->bV += d_bV; st->bJ += d_bJ; st->M += d_M; st->Ms += d_Ms;
      st->n_attempt += d_att; st->n_accept += d_acc; st->n_null += d_null;
    }
    orc_measure(st, trace ? trace + 6 * s : NULL);
    st->sweep += 1;
  }
  return 0;
}

/* S0 "sequential random pairs": the literal algorithm of sec. 3.1 with a
 * completely random choice of the coupled pair, any Lx x Ly.
 * floor(N/2) pair updates per sweep.                                          */
int orc_sweep_s0(orc_state* st, int8_t* code, double T, int64_t nsweeps, int64_t* trace) {
  int64_t N = (int64_t)st->Lx * st->Ly;
  if (N < 2) return -1;
  if (!(T > 0.0)) return -2;
  for (int64_t s = 0; s < nsweeps; ++s) {
    for (int64_t k = 0; k < N / 2; ++k) {
      uint32_t w[4];
      orc_philox_tagged(st->seed, (uint32_t)k, 0, (uint32_t)st->sweep, (uint32_t)st->replica, TAG_S0, w);
      int64_t a = (int64_t)(((uint64_t)w[2] * (uint64_t)N) >> 32);
      int64_t b = (int64_t)(((uint64_t)w[3] * (uint64_t)(N - 1)) >> 32);
      if (b >= a) ++b;
      orc_pair_update(st, code, (int)(a % st->Lx), (int)(a / st->Lx), (int)(b % st->Lx), (int)(b / st->Lx), w[0], T);
    }
    orc_measure(st, trace ? trace + 6 * s : NULL);
    st->sweep += 1;
  }
  return 0;
}
