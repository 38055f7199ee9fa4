/*
 * oracle/ic_enum.c -- exact enumeration of tiny lattices.  TEST INFRASTRUCTURE.
 *
 * The paper validates every implementation against the exact solution of the
 * 4x4 lattice (sec. 3.3); its numbers are only in figures that are
 * not available, so the exact constrained canonical ensemble is rebuilt here by
 * enumeration.  Two independent routes:
 *
 *   orc_enum_bruteforce : odometer over all 4^N states, every state evaluated by
 *                         orc_recompute (eq. 3 written out).  N <= 12.
 *   orc_enum_rows       : row decomposition (states of one row tabulated, rows
 *                         combined), used for 4x4 (2^32 states).  Checked against
 *                         the brute force on 3x3 / 2x4 / 4x2 / 3x4 in the tests,
 *                         and against the closed form C(2N, N+Q) for the number
 *                         of states per charge sector.
 *
 * Output: a density of states, i.e. the number of states per key.  Everything
 * else (<E>, <E^2>, C(T), ...) is formed from it in Python (oracle/exact.py).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include "ic_oracle.h"

static const int S_OF[4] = {0, 0, +1, -1};
static const int SG_OF[4] = {+1, -1, 0, 0};

/* keys: (n2, bV, bJ, M, Ms, Q) as returned by orc_recompute.  Open-addressing
 * hash on the 6-tuple.  Returns the number of distinct keys, or -1 if cap is
 * too small / N too large.                                                    */
int64_t orc_enum_bruteforce(int Lx, int Ly, int64_t* keys, uint64_t* counts, int64_t cap) {
  int N = Lx * Ly;
  if (N < 1 || N > 12) return -1;
  int64_t hcap = 1;
  while (hcap < 4 * cap) hcap <<= 1;
  int64_t* slot = (int64_t*)malloc(sizeof(int64_t) * (size_t)hcap);
  if (!slot) return -1;
  for (int64_t i = 0; i < hcap; ++i) slot[i] = -1;
  int64_t nkeys = 0;
  int8_t code[16];
  uint64_t total = 1ull << (2 * N);
  for (uint64_t s = 0; s < total; ++s) {
    for (int i = 0; i < N; ++i) code[i] = (int8_t)((s >> (2 * i)) & 3);
    int64_t k6[6];
    orc_recompute(code, Lx, Ly, k6);
    uint64_t h = 1469598103934665603ull;
    for (int i = 0; i < 6; ++i) { h ^= (uint64_t)(k6[i] + 1000); h *= 1099511628211ull; }
    int64_t p = (int64_t)(h & (uint64_t)(hcap - 1));
    for (;;) {
      if (slot[p] < 0) {
        if (nkeys >= cap) { free(slot); return -1; }
        slot[p] = nkeys;
        memcpy(keys + 6 * nkeys, k6, sizeof k6);
        counts[nkeys] = 1;
        ++nkeys;
        break;
      }
      if (memcmp(keys + 6 * slot[p], k6, sizeof k6) == 0) { counts[slot[p]] += 1; break; }
      p = (p + 1) & (hcap - 1);
    }
  }
  free(slot);
  return nkeys;
}

/* Row decomposition.  A row state r is Lx site codes (2 bits each).  Tabulated
 * per row: charge q, n2, horizontal bonds hV/hJ (periodic in x: site x with
 * x+1 mod Lx, so Lx = 2 gives a double bond), magnetisation m and the row's
 * x-staggered magnetisation ms = sum_x (-1)^x sigma_x.  Tabulated per ordered
 * pair of rows: vertical bonds vV/vJ.  A lattice state is (r_0..r_{Ly-1});
 * vertical bonds join row y with row y+1 mod Ly.
 * keys: (Q, n2, bV, bJ); per key also the sums of M^2 and Ms^2 over the states
 * of that key.  Dense accumulation, then compaction.  Lx <= 4, Ly <= 4.        */
int64_t orc_enum_rows(int Lx, int Ly, int nthreads, int64_t* keys, uint64_t* counts,
                      uint64_t* sumM2, uint64_t* sumMs2, int64_t cap) {
  if (Lx < 1 || Lx > 4 || Ly < 1 || Ly > 4) return -1;
  const int R = 1 << (2 * Lx);
  const int N = Lx * Ly;
  int* q = malloc(sizeof(int) * R); int* n2 = malloc(sizeof(int) * R);
  int* hV = malloc(sizeof(int) * R); int* hJ = malloc(sizeof(int) * R);
  int* m = malloc(sizeof(int) * R); int* ms = malloc(sizeof(int) * R);
  int8_t* vV = malloc((size_t)R * R); int8_t* vJ = malloc((size_t)R * R);
  for (int r = 0; r < R; ++r) {
    int c[4];
    for (int x = 0; x < Lx; ++x) c[x] = (r >> (2 * x)) & 3;
    q[r] = n2[r] = hV[r] = hJ[r] = m[r] = ms[r] = 0;
    for (int x = 0; x < Lx; ++x) {
      int xr = (x + 1) % Lx;
      q[r] += S_OF[c[x]]; n2[r] += S_OF[c[x]] * S_OF[c[x]];
      hV[r] += S_OF[c[x]] * S_OF[c[xr]]; hJ[r] += SG_OF[c[x]] * SG_OF[c[xr]];
      m[r] += SG_OF[c[x]]; ms[r] += ((x & 1) ? -1 : 1) * SG_OF[c[x]];
    }
  }
  for (int r = 0; r < R; ++r)
    for (int t = 0; t < R; ++t) {
      int v = 0, j = 0;
      for (int x = 0; x < Lx; ++x) {
        int a = (r >> (2 * x)) & 3, b = (t >> (2 * x)) & 3;
        v += S_OF[a] * S_OF[b]; j += SG_OF[a] * SG_OF[b];
      }
      vV[(size_t)r * R + t] = (int8_t)v; vJ[(size_t)r * R + t] = (int8_t)j;
    }
  /* dense index: Q in [-N,N], n2 in [0,N], bV,bJ in [-2N,2N] */
  const int64_t dQ = 2 * N + 1, dn = N + 1, db = 4 * N + 1;
  const int64_t dense = dQ * dn * db * db;
  if (nthreads < 1) nthreads = 1;
  uint64_t* acc = calloc((size_t)(3 * dense) * (size_t)nthreads, sizeof(uint64_t));
  if (!acc) return -1;
  const int Rn[4] = {R, Ly > 1 ? R : 1, Ly > 2 ? R : 1, Ly > 3 ? R : 1};
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
  for (int r0 = 0; r0 < Rn[0]; ++r0) {
    int tid = 0;
#ifdef _OPENMP
    extern int omp_get_thread_num(void);
    tid = omp_get_thread_num();
#endif
    uint64_t* A = acc + (size_t)(3 * dense) * (size_t)tid;
    for (int r1 = 0; r1 < Rn[1]; ++r1)
      for (int r2 = 0; r2 < Rn[2]; ++r2)
        for (int r3 = 0; r3 < Rn[3]; ++r3) {
          int rows[4] = {r0, r1, r2, r3};
          int Q = 0, s2 = 0, bV = 0, bJ = 0, M = 0, Ms = 0;
          for (int y = 0; y < Ly; ++y) {
            int r = rows[y], t = rows[(y + 1) % Ly];
            Q += q[r]; s2 += n2[r]; bV += hV[r]; bJ += hJ[r]; M += m[r];
            Ms += ((y & 1) ? -1 : 1) * ms[r];
            bV += vV[(size_t)r * R + t]; bJ += vJ[(size_t)r * R + t];
          }
          int64_t idx = (((int64_t)(Q + N) * dn + s2) * db + (bV + 2 * N)) * db + (bJ + 2 * N);
          A[3 * idx] += 1; A[3 * idx + 1] += (uint64_t)(M * M); A[3 * idx + 2] += (uint64_t)(Ms * Ms);
        }
  }
  int64_t nkeys = 0;
  for (int64_t idx = 0; idx < dense; ++idx) {
    uint64_t c = 0, a = 0, b = 0;
    for (int t = 0; t < nthreads; ++t) {
      const uint64_t* A = acc + (size_t)(3 * dense) * (size_t)t;
      c += A[3 * idx]; a += A[3 * idx + 1]; b += A[3 * idx + 2];
    }
    if (!c) continue;
    if (nkeys >= cap) { nkeys = -1; break; }
    int64_t rem = idx;
    int64_t kJ = rem % db; rem /= db;
    int64_t kV = rem % db; rem /= db;
    int64_t k2 = rem % dn; rem /= dn;
    keys[4 * nkeys + 0] = rem - N; keys[4 * nkeys + 1] = k2;
    keys[4 * nkeys + 2] = kV - 2 * N; keys[4 * nkeys + 3] = kJ - 2 * N;
    counts[nkeys] = c; sumM2[nkeys] = a; sumMs2[nkeys] = b;
    ++nkeys;
  }
  free(acc); free(q); free(n2); free(hV); free(hJ); free(m); free(ms); free(vV); free(vJ);
  return nkeys;
}
