/*
 * oracle/ic_variants.c -- CPU ORACLE, part 2.  TEST INFRASTRUCTURE, NOT PRODUCT CODE (see ic_oracle.c).
 *
 * Plain, slow, step-by-step C for what the paper describes around its main algorithm:
 *
 *   orc_sweep_nn          the paper's FIRST version of the coupled-pair algorithm: "one site was randomly
 *                         selected, the other chosen among its neighbours" (Fig. 3), which it
 *                         found wrong at low temperature on 4x4 (no second heat-capacity peak).
 *   orc_sweep_mu          the method the paper replaces: single-site Metropolis with the extra energy term
 *                         -mu * sum_i S_i, mu adjusted automatically so that sum S stays near n N
 *                         (sec. 2.2), whose heat capacity diverges as T -> 0.
 *   orc_build_map_paper   "Algorithm for building a map", literally: L x L bool array,
 *                         rejection sampling of unmarked sites, marking of the pair's nearest neighbours.
 *   orc_build_map_luby    the same kind of map built without a sequential scan: K random candidate pairs, a
 *                         candidate survives iff no candidate of lower index has a site inside its covering
 *                         (its two sites and their neighbours, Fig. 1).  This is what the CUDA
 *                         library builds on the device (ic_sweep_maps); DESIGN.md "Maps".
 *   orc_sweep_maps        sweeps made of such maps: every pair of a map gets one coupled-pair update
 *                         (PAPER.md:133), the same map for every lattice copy.
 *   orc_largest_cluster   size of the largest connected cluster of charged sites (the "drop" of PAPER.md:161-163,
 *                         Fig. 7), 4-neighbour connectivity, periodic.
 *
 * Parity pins (tests/test_oracle_variants.py):
 *   orc_sweep_nn, orc_sweep_maps   exact <E>, <E^2> of the enumerated 4x4 / 3x3 ensembles at high T (they are valid
 *                                  Markov chains for eq. 2+3); maps: conflict-freeness (V2) by brute force
 *   orc_sweep_mu at fixed mu       exact grand-canonical averages from the enumerated density of states
 *   orc_build_map_luby             O(K^2) brute-force statement of the survival rule in the test
 *   orc_largest_cluster            brute-force flood fill in Python on small lattices, closed forms (stripes, blocks)
 *   the mu-adjustment rule and the map parameters (K, N/10) are ours where the paper is silent: "parity unpinned"
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include "ic_oracle.h"

static const int S_OF[4] = {0, 0, +1, -1};
static const int SG_OF[4] = {+1, -1, 0, 0};
enum { TAG_NN = 4, TAG_MU = 5, TAG_MAP = 6, TAG_MAPU = 7 };

static inline int wrap(int v, int L) { v %= L; return v < 0 ? v + L : v; }

/* ------------------------------------------------------------------------- */
/* Nearest-neighbour-only coupled pairs: floor(N/2) updates per  */
/* sweep; a = random site, b = one of its four neighbour slots at random.       */
/* ------------------------------------------------------------------------- */
int orc_sweep_nn(orc_state* st, int8_t* code, double T, int64_t nsweeps, int64_t* trace) {
  const int64_t N = (int64_t)st->Lx * st->Ly;
  static const int dx[4] = {+1, -1, 0, 0}, dy[4] = {0, 0, +1, -1};
  if (N < 2) return -1;
  if (!(T > 0.0)) return -2;
  for (int64_t s = 0; s < nsweeps; ++s) {
    for (int64_t k = 0; k < N / 2; ++k) {
      uint32_t w[4];
      orc_philox_tagged(st->seed, (uint32_t)k, 0, (uint32_t)st->sweep, (uint32_t)st->replica, TAG_NN, w);
      int64_t a = (int64_t)(((uint64_t)w[2] * (uint64_t)N) >> 32);
      int xa = (int)(a % st->Lx), ya = (int)(a / st->Lx), d = (int)(w[3] >> 30);
      int xb = wrap(xa + dx[d], st->Lx), yb = wrap(ya + dy[d], st->Ly);
      if (xb == xa && yb == ya) continue; /* a dimension of size 1 */
      orc_pair_update(st, code, xa, ya, xb, yb, w[0], T);
    }
    orc_measure(st, trace ? trace + 6 * s : NULL);
    st->sweep += 1;
  }
  return 0;
}

/* ------------------------------------------------------------------------- */
/* Penalty / chemical-potential method.  Single-site Metropolis */
/* on H = E - mu * sum S: N attempts per sweep, a random site proposes one of   */
/* the four states; after every sweep mu += kappa * (Q_target - sum S) / N      */
/* ("automatically adjusting the parameter mu"; the rule itself is ours: the    */
/* paper gives none).  The recorded energy is E of eq. (3), without the mu term.*/
/* trace rows: (n2, bV, bJ, M, Ms, Q) with the CURRENT sum S as Q.              */
/* ------------------------------------------------------------------------- */
int orc_sweep_mu(orc_state* st, int8_t* code, double T, int64_t nsweeps, double* mu, double kappa, int64_t q_target,
                 int64_t* trace) {
  const int Lx = st->Lx, Ly = st->Ly;
  const int64_t N = (int64_t)Lx * Ly;
  static const int dx[4] = {+1, -1, 0, 0}, dy[4] = {0, 0, +1, -1};
  if (!(T > 0.0)) return -2;
  for (int64_t s = 0; s < nsweeps; ++s) {
    for (int64_t k = 0; k < N; ++k) {
      uint32_t w[4];
      orc_philox_tagged(st->seed, (uint32_t)k, 0, (uint32_t)st->sweep, (uint32_t)st->replica, TAG_MU, w);
      int64_t i = (int64_t)(((uint64_t)w[2] * (uint64_t)N) >> 32);
      int x = (int)(i % Lx), y = (int)(i / Lx);
      int c = code[i], nc = (int)(w[0] & 3u);
      if (nc == c) continue;
      int nS = 0, nG = 0;
      for (int d = 0; d < 4; ++d) {
        int j = code[(int64_t)wrap(y + dy[d], Ly) * Lx + wrap(x + dx[d], Lx)];
        nS += S_OF[j]; nG += SG_OF[j];
      }
      /* eq. (3): the site's on-site term and its four bonds (a dimension of size 2 gives double bonds,
       * which the four neighbour slots count twice, as eq. (3) does) */
      int dS = S_OF[nc] - S_OF[c], dG = SG_OF[nc] - SG_OF[c];
      int dn2 = S_OF[nc] * S_OF[nc] - S_OF[c] * S_OF[c], dV = dS * nS, dJ = dG * nG;
      double dH = ((st->delta * (double)dn2 + st->V * (double)dV) + (0.25 * st->J) * (double)dJ) - (*mu) * (double)dS;
      if (dH > 0.0) {
        double u = (double)(w[1] >> 3) / 536870912.0;
        if (!(u < exp(-dH / T))) continue;
      }
      code[i] = (int8_t)nc;
      st->n2 += dn2; st->bV += dV; st->bJ += dJ; st->Q += dS;
      st->M += dG; st->Ms += (((x + y) & 1) ? -1 : +1) * dG;
    }
    *mu += kappa * (double)(q_target - st->Q) / (double)N;
    orc_measure(st, trace ? trace + 6 * s : NULL);
    st->sweep += 1;
  }
  return 0;
}

/* ------------------------------------------------------------------------- */
/* Maps                                                     */
/* ------------------------------------------------------------------------- */

/* The paper's algorithm, steps 1-7.  Random sites come from the stream
 * Philox(ctr = (j, 0, map_index, TAG_MAP)), four sites per block, in order.  Gives up after 64 N draws
 * (reading G11: the paper's "such a number of pairs must exist" is not guaranteed).  Returns the number
 * of pairs placed (<= npairs). */
int64_t orc_build_map_paper(int Lx, int Ly, uint64_t seed, uint64_t map_index, int64_t npairs, int64_t* ia, int64_t* ib) {
  const int64_t N = (int64_t)Lx * Ly;
  static const int dx[4] = {+1, -1, 0, 0}, dy[4] = {0, 0, +1, -1};
  uint8_t* mark = (uint8_t*)calloc((size_t)N, 1);                 /* step 1 */
  if (!mark) return -1;
  uint32_t w[4]; int have = 0; uint64_t blk = 0; int64_t draws = 0, placed = 0;
  int64_t pick[2];
  while (placed < npairs) {
    int got = 0;
    while (got < 2 && draws < 64 * N) {                            /* steps 2-4 */
      if (have == 0) { orc_philox_tagged(seed, (uint32_t)blk, (uint32_t)(blk >> 32), (uint32_t)map_index, 0, TAG_MAP, w); ++blk; have = 4; }
      int64_t s = (int64_t)(((uint64_t)w[4 - have] * (uint64_t)N) >> 32); --have; ++draws;
      if (mark[s]) continue;
      mark[s] = 1; pick[got++] = s;
    }
    if (got < 2) break;
    ia[placed] = pick[0]; ib[placed] = pick[1]; ++placed;         /* step 5 */
    for (int k = 0; k < 2; ++k) {                                   /* step 6 */
      int x = (int)(pick[k] % Lx), y = (int)(pick[k] / Lx);
      for (int d = 0; d < 4; ++d) mark[(int64_t)wrap(y + dy[d], Ly) * Lx + wrap(x + dx[d], Lx)] = 1;
    }
  }                                                                 /* step 7 */
  free(mark);
  return placed;
}

/* Candidate k of map `map_index`: a = (w0 N) >> 32, b = (w1 (N-1)) >> 32 skipping a, from
 * Philox(ctr = (k, 0, map_index, TAG_MAP)): two distinct uniformly random sites. */
static void map_candidate(int64_t N, uint64_t seed, uint64_t map_index, int64_t k, int64_t* a, int64_t* b) {
  uint32_t w[4];
  orc_philox_tagged(seed, (uint32_t)k, (uint32_t)((uint64_t)k >> 32), (uint32_t)map_index, 0, TAG_MAP, w);
  *a = (int64_t)(((uint64_t)w[0] * (uint64_t)N) >> 32);
  *b = (int64_t)(((uint64_t)w[1] * (uint64_t)(N - 1)) >> 32);
  if (*b >= *a) ++*b;
}

/* K candidates; candidate k survives iff no candidate j < k (surviving or not) has one of its two sites
 * inside k's covering = {a_k, b_k} and their nearest neighbours.  first[s] = lowest index of a candidate
 * with site s.  alive[k] = 0/1; ia, ib = all K candidates.  Returns the number of survivors.            */
int64_t orc_build_map_luby(int Lx, int Ly, uint64_t seed, uint64_t map_index, int64_t K, int64_t* ia, int64_t* ib, uint8_t* alive) {
  const int64_t N = (int64_t)Lx * Ly;
  static const int dx[5] = {0, +1, -1, 0, 0}, dy[5] = {0, 0, 0, +1, -1};
  int64_t* first = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  if (!first) return -1;
  for (int64_t s = 0; s < N; ++s) first[s] = K;
  for (int64_t k = 0; k < K; ++k) {
    map_candidate(N, seed, map_index, k, &ia[k], &ib[k]);
    if (first[ia[k]] > k) first[ia[k]] = k;
    if (first[ib[k]] > k) first[ib[k]] = k;
  }
  int64_t n = 0;
  for (int64_t k = 0; k < K; ++k) {
    int ok = 1;
    const int64_t site2[2] = {ia[k], ib[k]};
    for (int e = 0; e < 2 && ok; ++e) {
      int x = (int)(site2[e] % Lx), y = (int)(site2[e] / Lx);
      for (int d = 0; d < 5; ++d)
        if (first[(int64_t)wrap(y + dy[d], Ly) * Lx + wrap(x + dx[d], Lx)] < k) { ok = 0; break; }
    }
    alive[k] = (uint8_t)ok; n += ok;
  }
  free(first);
  return n;
}

/* nmaps maps, one measurement after each (the paper's "step").  mode 0: the paper's
 * sequential builder with npairs = K; mode 1: K candidates, survivors only.  The random word of pair
 * (candidate) k is word k & 3 of Philox(ctr = (k >> 2, 1, map_index, replica | TAG_MAPU)); pairs are
 * updated in index order (any order gives the same lattice: they do not interact).  The map index is
 * the state's sweep counter.  attempted, if given, receives the total number of pair updates.        */
int orc_sweep_maps(orc_state* st, int8_t* code, double T, int64_t nmaps, int mode, int64_t K, int64_t* trace, int64_t* attempted) {
  const int Lx = st->Lx, Ly = st->Ly;
  if (!(T > 0.0)) return -2;
  if (K < 1) return -1;
  int64_t* ia = (int64_t*)malloc((size_t)K * sizeof(int64_t));
  int64_t* ib = (int64_t*)malloc((size_t)K * sizeof(int64_t));
  uint8_t* alive = (uint8_t*)malloc((size_t)K);
  if (!ia || !ib || !alive) { free(ia); free(ib); free(alive); return -3; }
  int64_t att = 0;
  for (int64_t m = 0; m < nmaps; ++m) {
    int64_t np = K;
    if (mode == 0) { np = orc_build_map_paper(Lx, Ly, st->seed, st->sweep, K, ia, ib); memset(alive, 1, (size_t)K); }
    else orc_build_map_luby(Lx, Ly, st->seed, st->sweep, K, ia, ib, alive);
    for (int64_t k = 0; k < np; ++k) {
      if (!alive[k]) continue;
      uint32_t w[4];
      orc_philox_tagged(st->seed, (uint32_t)(k >> 2), 1, (uint32_t)st->sweep, (uint32_t)st->replica, TAG_MAPU, w);
      orc_pair_update(st, code, (int)(ia[k] % Lx), (int)(ia[k] / Lx), (int)(ib[k] % Lx), (int)(ib[k] / Lx), w[k & 3], T);
      ++att;
    }
    orc_measure(st, trace ? trace + 6 * m : NULL);
    st->sweep += 1;
  }
  if (attempted) *attempted = att;
  free(ia); free(ib); free(alive);
  return 0;
}

/* ------------------------------------------------------------------------- */
/* Largest connected cluster of charged sites (the "drop").  */
/* which = 0: sites with S != 0; 1: S = +1 only; 2: S = -1 only.  4-neighbour   */
/* connectivity, periodic.  Flood fill with an explicit stack.  out2 = (size of */
/* the largest cluster, number of clusters).                                   */
/* ------------------------------------------------------------------------- */
int orc_largest_cluster(const int8_t* code, int Lx, int Ly, int which, int64_t out2[2]) {
  const int64_t N = (int64_t)Lx * Ly;
  static const int dx[4] = {+1, -1, 0, 0}, dy[4] = {0, 0, +1, -1};
  uint8_t* seen = (uint8_t*)calloc((size_t)N, 1);
  int64_t* stack = (int64_t*)malloc((size_t)N * sizeof(int64_t));
  if (!seen || !stack) { free(seen); free(stack); return -1; }
  int64_t best = 0, ncl = 0;
  for (int64_t s0 = 0; s0 < N; ++s0) {
    int c0 = code[s0];
    int in0 = which == 0 ? (c0 >= 2) : which == 1 ? (c0 == 2) : (c0 == 3);
    if (!in0 || seen[s0]) continue;
    int64_t top = 0, size = 0;
    stack[top++] = s0; seen[s0] = 1;
    while (top > 0) {
      int64_t s = stack[--top]; ++size;
      int x = (int)(s % Lx), y = (int)(s / Lx);
      for (int d = 0; d < 4; ++d) {
        int64_t t = (int64_t)wrap(y + dy[d], Ly) * Lx + wrap(x + dx[d], Lx);
        int c = code[t];
        int in = which == 0 ? (c >= 2) : which == 1 ? (c == 2) : (c == 3);
        if (in && !seen[t]) { seen[t] = 1; stack[top++] = t; }
      }
    }
    if (size > best) best = size;
    ++ncl;
  }
  out2[0] = best; out2[1] = ncl;
  free(seen); free(stack);
  return 0;
}
