// ic_kernels_coop.cuh -- variant 5: single mid-size lattices (128 <= L <= 1024, config C3 of BASELINE.json) on the tiled
// layouts LAY_P16 / LAY_P2.
//
// A sweep of a 1024 x 1024 lattice is 2 x 262 144 pair updates: a third of a microsecond of arithmetic for the whole chip.
// With one launch per phase such a run is bound by launch and memory latency, not by any throughput.  Here ONE
// cooperative launch runs all the sweeps of an ic_sweep call on the whole GPU:
//   * the lattice stays in global memory (L2-resident: 1 MiB at most); the class tables and the per-lane move descriptors
//     of the staged kernels sit in shared memory for the whole launch (no table fill per phase);
//   * an item is FOUR coupled pairs (one 32-bit word of a 16-site plane vector, one Philox block): 65 536 items per phase at
//     L = 1024 for 148 x 448 item threads, so every thread has at most one short item per phase and the phase is one memory
//     latency + one Philox block + one pairs4 (the item code of the staged kernels) long;
//   * the two phases of a sweep are separated by a barrier over the blocks of the replica (a counter in global memory:
//     red.release + ld.acquire poll);
//   * every block carries one service warp besides its item threads: while those are in phase 0 of sweep s it derives the
//     schedule of sweep s+1 (the Philox call the host makes) and adds the block's sums of sweep s-1 (per-thread sums -> warp
//     REDUX -> shared memory) into an accumulator in the workspace that is double buffered by the sweep's parity; the
//     service warp of the replica's first block folds sweep s-1 (U5, the operations of k_fold in the same order) during
//     phase 1.  Nothing serial is left on the item threads' path: two barriers per sweep.
// grid = (blocks per replica, rows); a row of blocks takes the replicas row, row + rows, ... in turn (rows = min(replicas,
// number of SMs)); cooperative launch (all blocks co-resident).  k_resvec_sweeps (below) runs the same items on a lattice
// resident in shared memory, one block per replica, for 16 <= L <= 64.
#pragma once
#include "ic_common.cuh"
#include "ic_kernels_ref.cuh"
#include "ic_kernels_p16.cuh"
#include "ic_kernels_staged.cuh"

namespace ic {

constexpr int COOP_THREADS = 512;
constexpr int COOP_MIN_L = 128, COOP_MAX_L = 1024;
constexpr int COOP_OFF_THR = 0;                                    // uint32 threshold[THR_STRIDE], packed deltas[THR_STRIDE]
constexpr int COOP_OFF_DESC = COOP_OFF_THR + THR_STRIDE * 8;       // [2 sweep types] uint2 descriptors [8][28][16]
constexpr int COOP_SMEM_BYTES = COOP_OFF_DESC + 2 * ST_DESC_SMEM;

struct CoopScratch {            // one per replica, in the workspace; set up before every launch: acc = 0, arrived = COOP_BAR_BASE
  long long acc[2][5];          // per-sweep sums (dn2, dV, dJ, M, Ms of the updated sites), buffer = sweep parity
  unsigned int arrived;         // barrier counter of the replica's blocks: + gridDim.x per barrier, modulo 2^32
  unsigned int pad[11];
};
static_assert(sizeof(CoopScratch) == 128, "CoopScratch layout");
// The counter grows by gridDim.x at each of the 2 nsweeps + 1 barriers of a launch and ic_sweep accepts up to 2^31 sweeps, so
// it wraps in a long call (148 blocks: after 14.5 M sweeps).  The barrier therefore compares modulo 2^32 (a block is never
// more than one barrier = gridDim.x < 2^31 counts away from the counter), and the counter STARTS one count below 2^32: every
// launch, hence every test of this kernel, crosses the wrap at its first barrier.
constexpr unsigned int COOP_BAR_BASE = 0xFFFFFFFFu;

struct CoopArgs {
  void* lattice; const uint2* thr; const uint2* desc32; ReplicaObs* obs; CoopScratch* scratch;
  long long* trace;              // nullptr or [nsweeps][replicas][6]
  long long lat_stride, nsweeps;
  unsigned long long sweep0;
  double delta, V, quarterJ;
  int L, logL, replicas;
  uint32_t key0, key1;
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// barrier over the blocks that share `counter`; everything the blocks wrote before it is visible to all of them after it
__device__ __forceinline__ void coop_barrier(unsigned int* counter, unsigned int target) {
  __syncthreads();                 // the block's writes happen before thread 0's release (causality order through the barrier)
  if (threadIdx.x == 0) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
    while ((int)(ld_acquire_u32(counter) - target) < 0) { }      // modulo 2^32: correct across the wrap of the counter
  }
  __syncthreads();
}

// the four site bytes at plane columns X .. X+3 (X a multiple of 4) of the plane row at site offset `row`
template <int BITS>
__device__ __forceinline__ uint32_t ldw(const uint8_t* lat, int row, int X) {
  if (BITS == 8) return *reinterpret_cast<const uint32_t*>(lat + row + X);
  const uint32_t w = *reinterpret_cast<const uint32_t*>(lat + ((row + (X & ~15)) >> 2));
  return __funnelshift_r(w, w, (X >> 1) & 6) & 0x09090909u;             // sites 4j .. 4j+3 of the word: rotr by 2j
}
// ... at X + sh .. X + sh + 3, sh in {-1, 0, +1}, periodic in the row of W sites (one tile per row quad)
template <int BITS>
__device__ __forceinline__ uint32_t ldw_sh(const uint8_t* lat, int row, int X, int W, int sh) {
  const uint32_t w = ldw<BITS>(lat, row, X);
  if (sh < 0) return (w << 8) | ldsite<BITS>(lat, row + ((X - 1) & (W - 1)));
  if (sh > 0) return (w >> 8) | (ldsite<BITS>(lat, row + ((X + 4) & (W - 1))) << 24);
  return w;
}

// stores the four site bytes `w4` (clean: bits 0 and 3) of word j of the vector at X0 of plane row `row`.
// P2: the four lanes of the quad merge their words and lane j = 0 stores the packed word.
template <int BITS>
__device__ __forceinline__ void st_word(uint8_t* lat, int row, int X0, int j, uint32_t w4) {
  if (BITS == 8) { *reinterpret_cast<uint32_t*>(lat + row + X0 + 4 * j) = w4; return; }
  // (the item order keeps the row class uniform in a warp, so every lane of the warp is here)
  uint32_t p = __funnelshift_l(w4, w4, 2 * j);
  p |= __shfl_xor_sync(0xFFFFFFFFu, p, 1);
  p |= __shfl_xor_sync(0xFFFFFFFFu, p, 2);
  if (j == 0) *reinterpret_cast<uint32_t*>(lat + ((row + X0) >> 2)) = p;
}
// the same for a vector that starts one site to the left (sites X0-1+4j .. X0+2+4j, periodic): bytes cross word borders
template <int BITS>
__device__ __forceinline__ void st_word_left1(uint8_t* lat, int row, int X0, int W, int j, uint32_t w4, uint32_t old4) {
  if (BITS == 8) {
#pragma unroll
    for (int m = 0; m < 4; ++m) lat[row + ((X0 - 1 + 4 * j + m) & (W - 1))] = (uint8_t)((w4 >> (8 * m)) & 0xFFu);
    return;
  }
  // P2: xor the changes into the words (two lanes of different quads may share a word; xor commutes)
  const uint32_t d = w4 ^ old4;
  if (d == 0u) return;
  uint32_t own = 0u;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    const uint32_t e = (d >> (8 * m)) & 9u;
    const int k = 4 * j - 1 + m;                               // site inside the word at X0; -1 = site 15 of the word to the left
    if (k < 0) { if (e) atomicXor(reinterpret_cast<uint32_t*>(lat + ((row + ((X0 - 16) & (W - 1))) >> 2)), rotl32(e, p2_shift(15))); }
    else own |= rotl32(e, p2_shift(k));
  }
  if (own) atomicXor(reinterpret_cast<uint32_t*>(lat + ((row + X0) >> 2)), own);
}

// Item it of a phase -> (word of the plane row, plane selector hi, row class half, row quad Y).  The word index is the lowest
// field; then as many low bits of Y as it takes to fill a warp, so that (hi, half) -- which decide the branches taken and
// the shapes of the stores -- are uniform in a warp whenever the lattice is large enough (L >= 128).
__device__ __forceinline__ void item_coords(int it, int lw, int& wi, int& hi, int& half, int& Y) {
  const int lgw = lw - 2;                                            // log2(words per plane row)
  const int nlo = min(lw, lgw < 5 ? 5 - lgw : 0);
  wi = it & ((1 << lgw) - 1);
  hi = (it >> (lgw + nlo)) & 1; half = (it >> (lgw + nlo + 1)) & 1;
  Y = ((it >> (lgw + nlo + 2)) << nlo) | ((it >> lgw) & ((1 << nlo) - 1));
}

// One item = the four coupled pairs of word wi of a plane row (PAPER.md:64-98 through pairs4, the item code of the
// staged kernels): loads of the ten words (a, b, eight neighbours), one Philox block, the update, the stores, and the
// item's contribution to the sweep's sums.  lat: the replica's lattice in LAY_P16 (BITS = 8; global or shared memory) or
// LAY_P2 (BITS = 2), one tile per row quad (L <= 2048).
template <int BITS>
__device__ __forceinline__ void coop_item(uint8_t* lat, int lw, int type, int p1, int p2, int phase, int wi, int hi, int half, int Y,
                                          uint32_t c2, uint32_t c3, uint32_t key0, uint32_t key1, uint32_t s_desc,
                                          int& tn2, int& tV, int& tJ, int& tM, int& tMs) {
  const int W = 1 << lw, Wm = W - 1, Lm = 4 * W - 1;
  const int Xj = 4 * wi, X0 = Xj & ~15, j = wi & 3;                  // plane column of the item's first pair; its 16-site vector; word in it
  uint32_t A4, B4, EA4, EB4, c0;
  int a3 = 0, sgn, ya;
  // plane row kx of lattice row y (one tile per row quad: (y >> 2) * 16 + (y & 3) * 4 + kx = 4 y + kx plane rows of W sites)
  auto R = [lw](int y, int kx) -> int { return ((y << 2) + kx) << lw; };
  if (type == 0) {
    // ---- FAR: a = (even x, y), b = its partner (x ^ mx, y ^ my); eq. (4) ------------------------------------------
    const int mx = p1, my = p2;
    const int kxa = 2 * hi, kxb = kxa ^ (mx & 3);
    ya = 4 * Y + phase + 2 * half;
    const int yb = ya ^ my;
    // b in a's lane order: lane i <-> i ^ c, c = (mx >> 2) & 15: word j of the permuted vector is word j ^ (c >> 2)
    // of the partner chunk, its bytes permuted by c & 3
    const int jb = j ^ (((mx >> 2) & 15) >> 2), Xb0 = X0 ^ ((mx >> 2) & Wm & ~15), Xb = Xb0 + 4 * jb;
    const uint32_t selb = 0x3210u ^ (0x1111u * (uint32_t)((mx >> 2) & 3));
    const int ra = R(ya, kxa), rb = R(yb, kxb);
    A4 = ldw<BITS>(lat, ra, Xj);
    const uint32_t b0 = ldw<BITS>(lat, rb, Xb);
    EA4 = ldw_sh<BITS>(lat, R(ya, (kxa + 3) & 3), Xj, W, kxa == 0 ? -1 : 0) + ldw<BITS>(lat, R(ya, kxa + 1), Xj) +
          ldw<BITS>(lat, R((ya - 1) & Lm, kxa), Xj) + ldw<BITS>(lat, R((ya + 1) & Lm, kxa), Xj);
    const uint32_t eb0 = ldw<BITS>(lat, R(yb, kxb - 1), Xb) + ldw_sh<BITS>(lat, R(yb, (kxb + 1) & 3), Xb, W, kxb == 3 ? 1 : 0) +
                         ldw<BITS>(lat, R((yb - 1) & Lm, kxb), Xb) + ldw<BITS>(lat, R((yb + 1) & Lm, kxb), Xb);
    B4 = __byte_perm(b0, 0u, selb); EB4 = __byte_perm(eb0, 0u, selb);
    c0 = (uint32_t)(4 * wi + kxa);
    const u32x4 rr = philox_update(c0, (uint32_t)ya, c2, c3, key0, key1);
    pairs4(A4, B4, EA4, EB4, rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, a3);
    st_word<BITS>(lat, ra, X0, j, A4);
    st_word<BITS>(lat, rb, Xb0, jb, __byte_perm(B4, 0u, selb));
    sgn = phase ? -2 : 2;                                            // both sites have the phase's colour
  } else if (p1 == 1) {
    // ---- NEAR, vertical dominoes: a = (x, y), b = the site below; eq. (5) ------------------------------------------
    const int kx = half + 2 * hi;
    ya = 4 * Y + ((p2 + 2 * ((half + phase) & 1)) & 3);
    const int yb = (ya + 1) & Lm;
    const int ra = R(ya, kx), rb = R(yb, kx);
    const int shl = kx == 0 ? -1 : 0, shr = kx == 3 ? 1 : 0;
    A4 = ldw<BITS>(lat, ra, Xj); B4 = ldw<BITS>(lat, rb, Xj);
    // vertical domino: a's lower neighbour is b, b's upper neighbour is a
    EA4 = ldw_sh<BITS>(lat, R(ya, (kx + 3) & 3), Xj, W, shl) + ldw_sh<BITS>(lat, R(ya, (kx + 1) & 3), Xj, W, shr) +
          ldw<BITS>(lat, R((ya - 1) & Lm, kx), Xj) + B4;
    EB4 = ldw_sh<BITS>(lat, R(yb, (kx + 3) & 3), Xj, W, shl) + ldw_sh<BITS>(lat, R(yb, (kx + 1) & 3), Xj, W, shr) +
          A4 + ldw<BITS>(lat, R((yb + 1) & Lm, kx), Xj);
    c0 = (uint32_t)(4 * wi + kx);
    const u32x4 rr = philox_update(c0, (uint32_t)ya, c2, c3, key0, key1);
    pairs4(A4, B4, EA4, EB4, rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, a3);
    st_word<BITS>(lat, ra, X0, j, A4);
    st_word<BITS>(lat, rb, X0, j, B4);
    sgn = ((kx + ya) & 1) ? -1 : 1;                                  // a and b have opposite colours
  } else {
    // ---- NEAR, horizontal dominoes of row y; lanes are indexed by the b-site; eq. (5) ------------------------------
    ya = 4 * Y + half + 2 * hi;
    const int ka = (p2 + 2 * ((half + phase) & 1)) & 3, kb = (ka + 1) & 3;
    const int sh_a = -(ka == 3), sh_l = sh_a - (ka == 0), sh_r = (kb == 3);
    const int yu = (ya - 1) & Lm, yd = (ya + 1) & Lm;
    const int ra = R(ya, ka), rb = R(ya, kb);
    A4 = ldw_sh<BITS>(lat, ra, Xj, W, sh_a); B4 = ldw<BITS>(lat, rb, Xj);
    EA4 = ldw_sh<BITS>(lat, R(ya, (ka + 3) & 3), Xj, W, sh_l) + B4 +
          ldw_sh<BITS>(lat, R(yu, ka), Xj, W, sh_a) + ldw_sh<BITS>(lat, R(yd, ka), Xj, W, sh_a);
    EB4 = A4 + ldw_sh<BITS>(lat, R(ya, (kb + 1) & 3), Xj, W, sh_r) + ldw<BITS>(lat, R(yu, kb), Xj) + ldw<BITS>(lat, R(yd, kb), Xj);
    const uint32_t A4old = A4;
    c0 = (uint32_t)(4 * wi + kb);
    const u32x4 rr = philox_update(c0, (uint32_t)ya, c2, c3, key0, key1);
    pairs4(A4, B4, EA4, EB4, rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, a3);
    st_word<BITS>(lat, rb, X0, j, B4);
    if (sh_a == 0) st_word<BITS>(lat, ra, X0, j, A4); else st_word_left1<BITS>(lat, ra, X0, W, j, A4, A4old);
    sgn = ((ka + ya) & 1) ? -1 : 1;
  }
  // M and Ms of the eight sites from their new bytes f | g<<3: sum sigma = sum f - sum g = (9 sum f - sum (f + 8 g)) / 8
  {
    const int Fa = __dp4a((int)(A4 & 0x07070707u), 0x01010101, 0), Fb = __dp4a((int)(B4 & 0x07070707u), 0x01010101, 0);
    const int Ma = (9 * Fa - __dp4a((int)A4, 0x01010101, 0)) >> 3, Mb = (9 * Fb - __dp4a((int)B4, 0x01010101, 0)) >> 3;
    tM += Ma + Mb;
    tMs += (sgn & 1) ? sgn * (Ma - Mb) : (sgn >> 1) * (Ma + Mb);
  }
  // unpack the item's sums: a3 = dJ + (dV << 11) + (dn2 << 22)
  const int j11 = (a3 << 21) >> 21; a3 = (a3 - j11) >> 11;
  const int v11 = (a3 << 21) >> 21; a3 = (a3 - v11) >> 11;
  tJ += j11; tV += v11; tn2 += a3;
}

// ---- pieces shared by the two one-launch kernels -------------------------------------------------------------------------
// class tables and per-lane move descriptors of both sweep types into shared memory (once per launch)
__device__ __forceinline__ void fill_item_tables(unsigned char* smem, uint32_t smem0, const uint2* thr_r, const uint2* desc32, int tid, int nthr) {
  uint32_t* thr_s = reinterpret_cast<uint32_t*>(smem + COOP_OFF_THR);
  for (int k = tid; k < THR_STRIDE; k += nthr) { const uint2 v = __ldg(&thr_r[k]); thr_s[k] = v.x; thr_s[THR_STRIDE + k] = v.y; }
  uint2* desc_s = reinterpret_cast<uint2*>(smem + COOP_OFF_DESC);
  for (int k = tid; k < 2 * ST_DESC_SMEM / 8; k += nthr) {
    const int adj = k >= ST_DESC_SMEM / 8, kk = adj ? k - ST_DESC_SMEM / 8 : k;
    const int row = kk >> 4, rr = row / 28, key = row - 28 * rr;
    uint2 d = __ldg(&desc32[adj * ST_DESC_ENTRIES + key * 8 + rr]);
    d.y += smem0 + COOP_OFF_THR;                // low 16 bits: shared-memory address of the class base
    desc_s[k] = d;
  }
}
// U4: parameters of a sweep, the same for all replicas (identical maps for all copies)
__device__ __forceinline__ void sweep_schedule(int L, unsigned long long sweep, uint32_t key0, uint32_t key1, int* par) {
  const u32x4 z = philox4x32_10(0u, 0u, (uint32_t)sweep, TAG_SCHED << 28, key0, key1);
  if ((sweep & 1) == 0) { par[0] = 0; par[1] = (int)(2 * (z.v[0] & (uint32_t)(L / 2 - 1)) + 1); par[2] = (int)(2 * (z.v[1] & (uint32_t)(L / 2 - 1)) + 1); }
  else { par[0] = 1; par[1] = (int)(z.v[0] & 1u); par[2] = (int)(z.v[1] & 3u); }
}
// U5 for one sweep: the integers are current; one rounding per operation, the order of k_fold
__device__ __forceinline__ void fold_sweep(ReplicaObs& o, double delta, double V, double quarterJ, long long* trace_row) {
  const double E = __dadd_rn(__dadd_rn(__dmul_rn(delta, (double)o.n2), __dmul_rn(V, (double)o.bV)), __dmul_rn(quarterJ, (double)o.bJ));
  const double M = (double)o.M, Ms = (double)o.Ms;
  o.sumE = __dadd_rn(o.sumE, E); o.sumE2 = __dadd_rn(o.sumE2, __dmul_rn(E, E));
  o.sumM = __dadd_rn(o.sumM, M); o.sumM2 = __dadd_rn(o.sumM2, __dmul_rn(M, M)); o.sumAbsM = __dadd_rn(o.sumAbsM, fabs(M));
  o.sumMs = __dadd_rn(o.sumMs, Ms); o.sumMs2 = __dadd_rn(o.sumMs2, __dmul_rn(Ms, Ms)); o.sumAbsMs = __dadd_rn(o.sumAbsMs, fabs(Ms));
  o.nmeas += 1;
  if (trace_row) { trace_row[0] = o.n2; trace_row[1] = o.bV; trace_row[2] = o.bJ; trace_row[3] = o.M; trace_row[4] = o.Ms; trace_row[5] = o.Q; }
}
// the warp's sums of a sweep -> red[k][warp]
__device__ __forceinline__ void warp_sums(int (*red)[COOP_THREADS / 32], int warp, int lane, int tn2, int tV, int tJ, int tM, int tMs) {
  const unsigned full = 0xFFFFFFFFu;
  tn2 = __reduce_add_sync(full, tn2); tV = __reduce_add_sync(full, tV); tJ = __reduce_add_sync(full, tJ);
  tM = __reduce_add_sync(full, tM); tMs = __reduce_add_sync(full, tMs);
  if (lane == 0) { red[0][warp] = tn2; red[1][warp] = tV; red[2][warp] = tJ; red[3][warp] = tM; red[4][warp] = tMs; }
}

// Both kernels run blockDim.x - 32 item threads and one SERVICE WARP (the last) that keeps everything serial off the
// item threads' path: while they are in phase 0 of sweep s, its lane 0 derives the schedule of sweep s+1 and the warp adds up
// the block's sums of sweep s-1 (written to red[(s-1)&1] before the barrier that ended that sweep); the fold of sweep s-1
// (U5) follows.  All threads meet at the same barriers, two per sweep.
template <int BITS>
__global__ void __launch_bounds__(COOP_THREADS, 1) k_coop_sweeps(const CoopArgs A) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ int s_par[2][4];
  __shared__ int red[2][5][COOP_THREADS / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nit = (int)blockDim.x - 32;
  const bool service = tid >= nit;
  const uint32_t smem0 = smem_u32(smem);
  const int L = A.L, lw = A.logL - 2;
  const int n_items = 1 << (2 * lw);                               // (row quad, half, hi, word of the plane row): N/16 items of 4 pairs
  // a row of blocks (blockIdx.y) takes the replicas blockIdx.y, blockIdx.y + gridDim.y, ... one after the other, each for
  // all the sweeps of the call (replicas are independent; more replicas than SMs is the only case with more than one)
  for (int r = blockIdx.y; r < A.replicas; r += gridDim.y) {
  __syncthreads();                                                 // the previous replica's tables are no longer read
  fill_item_tables(smem, smem0, A.thr + (long long)r * THR_STRIDE, A.desc32, tid, (int)blockDim.x);
  uint8_t* lat = reinterpret_cast<uint8_t*>(A.lattice) + (long long)r * A.lat_stride;
  CoopScratch* sc = &A.scratch[r];
  const uint32_t c3 = (uint32_t)r | (TAG_UPDATE << 28);
  const bool folder = blockIdx.x == 0 && tid == nit;              // lane 0 of the service warp of the replica's first block
  ReplicaObs o;
  if (folder) o = A.obs[r];
  if (tid == nit) sweep_schedule(L, A.sweep0, A.key0, A.key1, s_par[0]);
  unsigned int bar_target = COOP_BAR_BASE;
  __syncthreads();

  // sums of sweep q: block -> the replica's accumulator acc[q & 1] (service warp); accumulator -> integers -> fold (folder)
  auto push_sums = [&](long long q) {
    const unsigned full = 0xFFFFFFFFu;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const int v = __reduce_add_sync(full, lane < (nit >> 5) ? red[q & 1][k][lane] : 0);
      if (lane == 0 && v) atomicAdd((unsigned long long*)&sc->acc[q & 1][k], (unsigned long long)(long long)v);
    }
  };
  auto fold = [&](long long q) {
    volatile long long* va = sc->acc[q & 1];
    o.n2 += va[0]; o.bV += va[1]; o.bJ += va[2]; o.M = va[3]; o.Ms = va[4];      // the two phases covered every site once
    va[0] = 0; va[1] = 0; va[2] = 0; va[3] = 0; va[4] = 0;                       // next used for sweep q + 2, five barriers on
    fold_sweep(o, A.delta, A.V, A.quarterJ, A.trace ? A.trace + 6LL * ((long long)A.replicas * q + r) : nullptr);
  };

  for (long long s = 0; s < A.nsweeps; ++s) {
    const unsigned long long sweep = A.sweep0 + (unsigned long long)s;
    const int type = s_par[s & 1][0], p1 = s_par[s & 1][1], p2 = s_par[s & 1][2];
    const uint32_t s_desc = smem0 + COOP_OFF_DESC + (type ? ST_DESC_SMEM : 0) + (uint32_t)(lane & 15) * 8u;
    int tn2 = 0, tV = 0, tJ = 0, tM = 0, tMs = 0;       // this thread's sums over both phases of the sweep
    for (int phase = 0; phase < 2; ++phase) {
      if (!service) {
        const uint32_t c2 = (uint32_t)(2 * sweep + (unsigned long long)phase);
        for (int it = blockIdx.x * nit + tid; it < n_items; it += gridDim.x * nit) {
          int wi, hi, half, Y;
          item_coords(it, lw, wi, hi, half, Y);
          coop_item<BITS>(lat, lw, type, p1, p2, phase, wi, hi, half, Y, c2, c3, A.key0, A.key1, s_desc, tn2, tV, tJ, tM, tMs);
        }
        if (phase == 1) warp_sums(red[s & 1], warp, lane, tn2, tV, tJ, tM, tMs);
      } else if (phase == 0) {
        if (lane == 0) sweep_schedule(L, sweep + 1, A.key0, A.key1, s_par[(s + 1) & 1]);
        if (s > 0) push_sums(s - 1);      // complete in every block before its arrival at the barrier below
      } else if (folder && s > 0) {
        fold(s - 1);                      // all blocks have passed the barrier after phase 0: the accumulator is complete
      }
      bar_target += gridDim.x;
      coop_barrier(&sc->arrived, bar_target);       // phase 1 reads neighbours written in phase 0, and the next sweep those of phase 1
    }
  }
  // the last sweep's sums
  if (A.nsweeps > 0) {
    if (service) push_sums(A.nsweeps - 1);
    bar_target += gridDim.x;
    coop_barrier(&sc->arrived, bar_target);
    if (folder) fold(A.nsweeps - 1);
  }
  if (folder) A.obs[r] = o;
  }   // replicas of this row of blocks
}

// ---------------------------------------------------------------------------------------------------------------
// Small lattices (16 <= L <= 64, configs C1 and C2): the same items with the replica's lattice resident in shared memory.
// One block per replica runs all the sweeps of an ic_sweep call; the lattice is converted from its layout in global memory
// (LAYG: ROW8, ROW2 or P16) to P16 bytes on the way in and back on the way out, the phases are separated by
// __syncthreads, lane 0 of the service warp folds sweep s-1 (U5) while the item threads are in phase 0 of sweep s.
// ---------------------------------------------------------------------------------------------------------------
constexpr int RESV_MIN_L = 16, RESV_MAX_L = 64;
constexpr int RESV_OFF_LAT = COOP_SMEM_BYTES;
constexpr int RESV_SMEM_BYTES = RESV_OFF_LAT + RESV_MAX_L * RESV_MAX_L;

template <int LAYG>
__global__ void __launch_bounds__(COOP_THREADS, 1) k_resvec_sweeps(const CoopArgs A) {
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ int s_par[2][4];
  __shared__ int red[2][5][COOP_THREADS / 32];
  const int r = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = (int)blockDim.x, nit = nthr - 32;
  const bool service = tid >= nit;
  const uint32_t smem0 = smem_u32(smem);
  const int L = A.L, logL = A.logL, lw = logL - 2, N = L * L;
  const LatView gv{(char*)A.lattice + (long long)r * A.lat_stride, L, logL};
  uint8_t* lat = smem + RESV_OFF_LAT;
  fill_item_tables(smem, smem0, A.thr + (long long)r * THR_STRIDE, A.desc32, tid, nthr);
  for (int i = tid; i < N; i += nthr) {
    const int x = i & (L - 1), y = i >> logL;
    lat[p16_site(lw, x, y)] = (uint8_t)e_of_code(Sites<LAYG>::load(gv, x, y));
  }
  const int n_items = 1 << (2 * lw);
  const uint32_t c3 = (uint32_t)r | (TAG_UPDATE << 28);
  ReplicaObs o;
  if (tid == nit) { o = A.obs[r]; sweep_schedule(L, A.sweep0, A.key0, A.key1, s_par[0]); }
  __syncthreads();

  auto fold = [&](long long q) {          // lane 0 of the service warp: block sums of sweep q -> integers -> U5
    long long M = 0, Ms = 0;
    for (int wv = 0; wv < (nit >> 5); ++wv) { o.n2 += red[q & 1][0][wv]; o.bV += red[q & 1][1][wv]; o.bJ += red[q & 1][2][wv]; M += red[q & 1][3][wv]; Ms += red[q & 1][4][wv]; }
    o.M = M; o.Ms = Ms;                   // the two phases covered every site once
    fold_sweep(o, A.delta, A.V, A.quarterJ, A.trace ? A.trace + 6LL * ((long long)A.replicas * q + r) : nullptr);
  };

  for (long long s = 0; s < A.nsweeps; ++s) {
    const unsigned long long sweep = A.sweep0 + (unsigned long long)s;
    const int type = s_par[s & 1][0], p1 = s_par[s & 1][1], p2 = s_par[s & 1][2];
    const uint32_t s_desc = smem0 + COOP_OFF_DESC + (type ? ST_DESC_SMEM : 0) + (uint32_t)(lane & 15) * 8u;
    int tn2 = 0, tV = 0, tJ = 0, tM = 0, tMs = 0;
    for (int phase = 0; phase < 2; ++phase) {
      if (!service) {
        const uint32_t c2 = (uint32_t)(2 * sweep + (unsigned long long)phase);
        for (int it = tid; it < n_items; it += nit) {
          int wi, hi, half, Y;
          item_coords(it, lw, wi, hi, half, Y);
          coop_item<8>(lat, lw, type, p1, p2, phase, wi, hi, half, Y, c2, c3, A.key0, A.key1, s_desc, tn2, tV, tJ, tM, tMs);
        }
        if (phase == 1) warp_sums(red[s & 1], warp, lane, tn2, tV, tJ, tM, tMs);
      } else if (phase == 0 && tid == nit) {
        sweep_schedule(L, sweep + 1, A.key0, A.key1, s_par[(s + 1) & 1]);
        if (s > 0) fold(s - 1);           // red[(s-1)&1] was complete at the barrier that ended sweep s-1; rewritten in sweep s+1
      }
      __syncthreads();       // phase 1 reads neighbours written in phase 0, and the next sweep those of phase 1
    }
  }
  if (tid == nit && A.nsweeps > 0) fold(A.nsweeps - 1);
  // the lattice goes back in its layout
  if (LAYG == LAY_ROW2) {
    uint32_t* words = reinterpret_cast<uint32_t*>(gv.base);
    for (int wi = tid; wi < (N >> 4); wi += nthr) {
      uint32_t wd = 0;
      const int y = (16 * wi) >> logL, x0 = (16 * wi) & (L - 1);
#pragma unroll
      for (int k = 0; k < 16; ++k) wd |= (uint32_t)code_of_e(lat[p16_site(lw, x0 + k, y)]) << (2 * k);
      words[wi] = wd;
    }
  } else if (LAYG == LAY_ROW8) {
    for (int i = tid; i < N; i += nthr) ((int8_t*)gv.base)[i] = (int8_t)code_of_e(lat[p16_site(lw, i & (L - 1), i >> logL)]);
  } else {
    for (int i = tid; i < N; i += nthr) ((uint8_t*)gv.base)[i] = lat[i];
  }
  if (tid == nit) A.obs[r] = o;
}

}  // namespace ic
