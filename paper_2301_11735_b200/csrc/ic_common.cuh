// ic_common.cuh -- definitions shared by the host control code and the sm_100a kernels of libic_b200.
//
// Notation follows the paper (arXiv:2301.11735): site state S = +-1 (charge) or s = +-1/2 with S = 0
// (magnetic), sigma = 2(1-S^2)s.  Public site code c: 0 sigma=+1, 1 sigma=-1, 2 S=+1, 3 S=-1.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#define IC_HD __host__ __device__ __forceinline__

namespace ic {

// ---------------------------------------------------------------------------------------------------
// Random numbers: Philox4x32 (Salmon, Moraes, Dror, Shaw, SC'11), counter-based, keyed by the seed.
// The paper only says pairs and configurations are "randomly selected"; U3.
// Counter = (c0, c1, c2, replica | tag << 28).
// ---------------------------------------------------------------------------------------------------
constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;
enum : uint32_t { TAG_UPDATE = 0, TAG_SCHED = 1, TAG_INIT = 2 };

struct u32x4 { uint32_t v[4]; };

IC_HD void mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
  const uint64_t p = (uint64_t)a * (uint64_t)b;   // one IMAD.WIDE on the device
  lo = (uint32_t)p; hi = (uint32_t)(p >> 32);
}

template <int ROUNDS>
IC_HD u32x4 philox4x32(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int round = 0; round < ROUNDS; ++round) {
    uint32_t h0, l0, h1, l1;
    mulhilo(PHILOX_M0, c0, h0, l0);
    mulhilo(PHILOX_M1, c2, h1, l1);
    c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
    k0 += PHILOX_W0; k1 += PHILOX_W1;
  }
  u32x4 r; r.v[0] = c0; r.v[1] = c1; r.v[2] = c2; r.v[3] = c3; return r;
}
// Schedule and stage-1 streams: the default ten rounds.  Update stream (one block per four pair updates, the hot path):
// Philox4x32-7, the seven-round member of the family that Salmon et al. report as the fewest rounds passing BigCrush
// (SURVEY 8(d) "RNG ladder", G5).
// Compile-time switch (G5 names the test that compares the sampled ensembles at 7 and 10 rounds): build with
// -DIC_PHILOX_UPDATE_ROUNDS=10 for the default
// member of the family; every kernel, the staged kernels' precomputed round keys included, follows this constant.
#ifndef IC_PHILOX_UPDATE_ROUNDS
#define IC_PHILOX_UPDATE_ROUNDS 7
#endif
constexpr int PHILOX_UPDATE_ROUNDS = IC_PHILOX_UPDATE_ROUNDS;
static_assert(PHILOX_UPDATE_ROUNDS >= 2 && PHILOX_UPDATE_ROUNDS <= 10, "the staged kernels precompute the first two rounds and ten round keys");
IC_HD u32x4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
  return philox4x32<10>(c0, c1, c2, c3, k0, k1);
}
IC_HD u32x4 philox_update(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
  return philox4x32<PHILOX_UPDATE_ROUNDS>(c0, c1, c2, c3, k0, k1);
}

// ---------------------------------------------------------------------------------------------------
// Site code -> S, sigma.  bit1 = "is a charge", bit0 = "negative".
// ---------------------------------------------------------------------------------------------------
IC_HD int S_of(int c) { return (c & 2) ? 1 - 2 * (c & 1) : 0; }
IC_HD int sg_of(int c) { return (c & 2) ? 0 : 1 - 2 * (c & 1); }

// ---------------------------------------------------------------------------------------------------
// Lattice layouts in device memory.
//   ROW8  one byte per site, public code, row-major [y][x]                       (8 bits/site, L < 64)
//   ROW2  2 bits per site, public code, 16 sites per 32-bit word, row-major       (2 bits/site)
//   P16   one byte per site, tiled: the lattice is cut into tiles of 4 rows x 4*SEGL columns (SEGL = min(L/4, 512));
//         a tile is stored contiguously as 16 "plane rows" [y&3][x&3] of SEGL bytes (plane column X = x>>2 inside the
//         tile), tiles in the order [X / SEGL][y>>2]: the tiles above and below a tile are its neighbours in memory, so
//         a tile with the plane rows of the lattice row above and below is ONE contiguous piece (one bulk copy).  Byte e = f | g<<3 with (f,g) = sigma+ (1,0), sigma- (0,1),
//         S+ (1,1), S- (0,0), so that the byte-wise sum of the four neighbour bytes is F | G<<3 with
//         sum S = F+G-4,  sum sigma = F-G                                          (8 bits/site, L >= 64)
//   P2    two bits per site, the tiles and plane rows of P16 with 16 plane sites per 32-bit word       (2 bits/site, L >= 128)
//         (a plane row of SEGL sites is SEGL/4 bytes, every byte offset of P16 divided by 4).  Site k = 4j + m of a word
//         keeps f at bit 8m + 2j and g at bit (8m + 2j + 3) mod 32, so that the four bytes f | g<<3 of the sites 4j .. 4j+3
//         are rotr(word, 2j) & 0x09090909: a word widens to the 16-byte vector the P16 arithmetic works on in
//         1 + 3 x 2 instructions and packs back in 5 (the residues {0,3}, {2,5}, {4,7}, {6,1} tile Z_8).
// Every phase of schedule S1 updates whole plane rows of P16 / P2, so the kernels work on dense 16-site vectors, and a
// tile (8 KB at SEGL = 512; 2 KB in P2) plus its neighbour rows is what one bulk copy stages in shared memory.
// ---------------------------------------------------------------------------------------------------
enum Layout : int { LAY_ROW8 = 0, LAY_ROW2 = 1, LAY_P16 = 2, LAY_P2 = 3 };

IC_HD int e_of_code(int c) { return (~c & 1) | (((c ^ (c >> 1)) & 1) << 3); }
IC_HD int code_of_e(int e) { int b0 = ~e & 1; return b0 | ((((e >> 3) ^ b0) & 1) << 1); }

// P16 addressing: lw = log2(L/4); byte offset of plane row (ky, kx) of tile (Y, seg)
constexpr int P16_LOGSEG_MAX = 9;
IC_HD int p16_logseg(int lw) { return lw < P16_LOGSEG_MAX ? lw : P16_LOGSEG_MAX; }
IC_HD long long p16_row(int lw, int ky, int kx, int Y, int seg) {
  const int ls = p16_logseg(lw);
  return ((((long long)seg << lw) + Y) * 16 + (ky * 4 + kx)) << ls;
}
IC_HD long long p16_site(int lw, int x, int y) {
  const int ls = p16_logseg(lw), X = x >> 2;
  return p16_row(lw, y & 3, x & 3, y >> 2, X >> ls) + (X & ((1 << ls) - 1));
}

// P2 words: bit position of site k's f inside its word; its g sits three bits on (mod 32)
IC_HD int p2_shift(int k) { return 8 * (k & 3) + 2 * (k >> 2); }
IC_HD uint32_t rotr32(uint32_t v, int s) { s &= 31; return s ? (v >> s) | (v << (32 - s)) : v; }
IC_HD uint32_t rotl32(uint32_t v, int s) { s &= 31; return s ? (v << s) | (v >> (32 - s)) : v; }
IC_HD int p2_site_e(uint32_t word, int k) { return (int)(rotr32(word, p2_shift(k)) & 9u); }   // byte f | g<<3 of site k
IC_HD long long p2_word(int lw, int x, int y) {        // byte offset of the word that holds site (x, y)
  const int ls = p16_logseg(lw), X = x >> 2;
  return (p16_row(lw, y & 3, x & 3, y >> 2, X >> ls) >> 2) + (((X & ((1 << ls) - 1)) >> 4) << 2);
}

struct LatView {              // one replica
  char* base;
  int L, logL;
};

template <int LAY>
struct Sites {
  static __device__ __forceinline__ long long p16_offset(const LatView& v, int x, int y) {
    return p16_site(v.logL - 2, x, y);
  }
  static __device__ __forceinline__ int load(const LatView& v, int x, int y) {
    if (LAY == LAY_P16) return code_of_e(((const uint8_t*)v.base)[p16_offset(v, x, y)]);
    if (LAY == LAY_P2) return code_of_e(p2_site_e(*(const uint32_t*)(v.base + p2_word(v.logL - 2, x, y)), (x >> 2) & 15));
    const long long i = ((long long)y << v.logL) + x;
    if (LAY == LAY_ROW8) return ((const int8_t*)v.base)[i];
    return (((const uint32_t*)v.base)[i >> 4] >> (2 * (int)(i & 15))) & 3;
  }
  // Sites written in one phase are distinct; with ROW2 / P2 several threads share a word: xor the change in.
  static __device__ __forceinline__ void store(const LatView& v, int x, int y, int oldc, int newc) {
    if (LAY == LAY_P16) { ((uint8_t*)v.base)[p16_offset(v, x, y)] = (uint8_t)e_of_code(newc); return; }
    if (LAY == LAY_P2) {
      const uint32_t d = (uint32_t)(e_of_code(oldc) ^ e_of_code(newc));
      if (d) atomicXor((uint32_t*)(v.base + p2_word(v.logL - 2, x, y)), rotl32(d, p2_shift((x >> 2) & 15)));
      return;
    }
    const long long i = ((long long)y << v.logL) + x;
    if (LAY == LAY_ROW8) ((int8_t*)v.base)[i] = (int8_t)newc;
    else atomicXor(&((uint32_t*)v.base)[i >> 4], (uint32_t)(oldc ^ newc) << (2 * (int)(i & 15)));
  }
};

// Acceptance class of a move (E_Delta, E_V, E_J): dn2 in {-2,0,2}, dV, dJ in [-16,16].
constexpr int N_CLASSES = 3 * 33 * 33;   // 3267 (the public, dense order of ic_thresholds)
// Device order of the class tables: index = (dn2/2+1)*CLS_SA + (dV+16)*CLS_SB + (dJ+16).  The strides decide which
// shared-memory bank a class falls into; with the dense strides (33, 33*33) the frequent classes collide (bank = dn2/2 + dV
// + dJ mod 32); 35 spreads them (measured on equilibrated lattices: 2.25 -> 1.53 wavefronts per 32-lane lookup).
constexpr int CLS_SB = 35, CLS_SA = 33 * CLS_SB;
constexpr int THR_STRIDE = 3520;         // table entries per replica (>= 3 * CLS_SA, multiple of 64)
// Device table entry of a class: x = 8*t29 - 1 (the move is accepted iff w <= x, which is (w >> 3) < t29),
// y = packed (dn2, dV, dJ) = dJ + (dV << 11) + (dn2 << 22) for the per-thread observable accumulator.
IC_HD int pack_delta(int dn2, int dV, int dJ) { return dJ + dV * 2048 + dn2 * 4194304; }
IC_HD int class_index(int dn2, int dV, int dJ) { return (dn2 / 2 + 1) * CLS_SA + (dV + 16) * CLS_SB + (dJ + 16); }
// Proposals that change nothing (abs(q) = 2, the current configuration, words 6 and 7 of a q = 0 pair) get a class entry of
// their own with threshold 0: "never accepted" instead of "dE = 0, always accepted".  The lattice cannot tell the
// difference; the kernels can: such lanes then skip the predicated second lookup and the write of the (empty) change.
constexpr int NULL_CLASS = 3 * CLS_SA;   // first entry after the real classes; its bank holds no frequent class
static_assert(NULL_CLASS < THR_STRIDE, "the null entry lies inside the table");
IC_HD int class_index_public(int dn2, int dV, int dJ) { return ((dn2 / 2 + 1) * 33 + (dV + 16)) * 33 + (dJ + 16); }

// Per-replica record in device memory: exact integers, then the fp64 sums of U5.
struct ReplicaObs {
  long long n2, bV, bJ, M, Ms, Q;      // current exact integers (updated by the phase kernels)
  long long nmeas, pad0;
  double sumE, sumE2, sumM, sumM2, sumAbsM, sumMs, sumMs2, sumAbsMs;
  long long Mnext, Msnext;             // staged kernels: M and Ms of the sites updated so far in the current sweep
};
static_assert(sizeof(ReplicaObs) == 144, "ReplicaObs layout");

// Task counters of the staged kernels: TASK_CTR_STRIDE words per replica (a cache line of its own), word p = phase p of the
// sweep in progress; zeroed by ic_create and by k_fold after every sweep.
constexpr int TASK_CTR_STRIDE = 32;

// Parameters of one phase of one sweep (schedule S1, U4), the same for all replicas
// (precedent: identical maps for all lattice copies).
struct PhaseArgs {
  void* lattice;                 // [replicas][lat_stride bytes]
  const uint2* thr;              // [replicas][THR_STRIDE] (8*t29-1, packed deltas)
  const uint2* desc;             // move descriptors of this sweep type (tiled kernels), [28*8]
  const uint2* desc32;           // move descriptors (coefficients, info) of both sweep types (staged kernels), [2][256]
  ReplicaObs* obs;               // [replicas]
  unsigned int* task_ctr;        // staged kernels: task counter of this phase, one per replica (stride TASK_CTR_STRIDE)
  long long lat_stride;          // bytes per replica
  int L, logL;
  int type;                      // 0 FAR (partner = (x^mx, y^my)), 1 NEAR (dominoes)
  int p1, p2;                    // FAR: mx, my.  NEAR: orientation (0 horizontal, 1 vertical), offset 0..3
  int phase;                     // 0 or 1
  uint32_t c2;                   // 2*sweep + phase
  uint32_t key0, key1;           // Philox key = seed
  // staged kernels: the ten round keys (key + i * Weyl constants) and the launch-constant parts of the first two rounds
  uint32_t rk[20];
  uint32_t f0, f1, f2;           // hi(M1*c2) ^ rk[0];  lo(M1*c2);  lo(M1*c2) ^ rk[2]
};

}  // namespace ic
