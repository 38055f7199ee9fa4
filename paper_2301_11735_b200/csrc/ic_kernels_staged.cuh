// ic_kernels_staged.cuh -- variant 3: the production sm_100a kernels for L >= 2048 on the tiled layouts LAY_P16 (one byte per
// site, BITS = 8) and LAY_P2 (two bits per site, BITS = 2: the same tiles with 16 plane sites per 32-bit word; bulk copies move
// the packed regions, consumers widen a word to the 16-byte vector on load and pack on store).
//
// One launch = one phase of a sweep (schedule S1, U4), one persistent block per SM, launched as a programmatic
// dependent of the previous kernel of the stream (table fill and barrier set-up overlap that kernel's tail):
//   * 2 producer warps (the last two of the block), one per consumer group, stage "regions" of the lattice in shared
//     memory with 1-D bulk copies (cp.async.bulk, the TMA engine; completion on an mbarrier).  A region is one tile of
//     the layout (row quad Y, 512 plane columns: 16 plane rows) plus the plane rows of the lattice row above and of the one
//     (NEAR-V: two) below.  Tiles are stored in the order [segment][Y], so the whole region is ONE contiguous piece of
//     12 KB (NEAR-V: 14 KB) and one bulk copy (two at the periodic wrap Y = 0 / Y = W-1).  The few bytes read across the
//     left/right tile edge (the x-1 neighbour of plane 0 is plane 3 one byte to the left) are fetched by the producer's
//     lanes with plain loads, issued a task ahead, into a small side array.
//   * 16 consumer warps in 2 groups; group g processes tasks g, g+2, ... of the block and owns two stage slots
//     (double buffering; a slot goes back to the producers as soon as the items are in registers).  A task is two
//     regions = 4096 coupled pairs, a thread's item one 16-byte vector = 16 pairs.  In a FAR phase the two regions are
//     partners under (x^mx, y^my): every byte of both is loaded once and all pairs between them are updated.
//   * consumers read 16-byte vectors from shared memory (conflict-free LDS.128), do the pair updates (byte-SIMD
//     neighbour sums, move descriptors, dp4a class index, integer acceptance) and store the updated
//     vectors straight to global memory (128-bit stores).
// No thread of a phase reads a byte that another thread of the phase writes: all neighbours of active sites are
// inactive (V2); bytes of active plane rows that belong to other tasks are staged but never used.
#pragma once
#include "ic_common.cuh"
#include "ic_kernels_ref.cuh"
#include "ic_kernels_p16.cuh"

namespace ic {

// Two groups of eight consumer warps: 18 warps per SM leave each thread the ~90 registers the item code wants (three groups at 72
// registers: -1.5 % at C5, -2.7 % at C4; measured, profiles/r02d)
constexpr int ST_GROUPS = 2;                  // consumer groups per block
constexpr int ST_DEPTH = 2;                   // ring slots per consumer group
constexpr int ST_NPROD = ST_GROUPS;           // producer warps per block: one per consumer group
constexpr int ST_LOGSEG = P16_LOGSEG_MAX, ST_SEG = 1 << ST_LOGSEG;   // plane columns per region = per tile of the layout
constexpr int ST_TPG = ST_SEG / 2;            // consumer threads per group: one 16-pair item each per task
constexpr int ST_CONS = ST_GROUPS * ST_TPG;   // consumer threads (warps 0..15); the producers are warps 16, 17
constexpr int ST_THREADS = ST_CONS + 32 * ST_NPROD;
constexpr int ST_DESC_ENTRIES = 256;          // move descriptors [key*8 + r] (224 used) in global memory: (coefficients, info)
constexpr int ST_DESC_SMEM = 28 * 8 * 128;    // in shared memory: [r][key][lane & 15] x 8 bytes, a private copy per lane
constexpr uint32_t ST_DESC_RSTRIDE = 28 * 128;

// What the consumers of one sub-task (region U, half) need to know about the task in a stage.
struct SubMeta {
  unsigned long long pa;     // global address of the a-side plane row (see the consumers)
  unsigned long long pb;     // global address of the b-side plane row
  unsigned long long pl;     // NEAR-H: address of the byte left of the a-side plane row (last byte of the tile to the left)
  int Y, C0;                 // row quad and first 16-column chunk of the sub-task's region (Philox counters)
};
static_assert(sizeof(SubMeta) == 32, "SubMeta layout");

template <int TYPE, int BITS>
struct StagedCfg {
  static constexpr int ROWS = TYPE == PH_NEAR_V ? 28 : 24;          // staged plane rows: (ky_rel + 1) * 4 + kx, ky_rel = -1..4 (5)
  static constexpr int RB = ST_SEG * BITS / 8;                      // bytes of a plane row of a tile: 512 (P16) or 128 (P2)
  static constexpr int REGION_BYTES = ROWS * RB;
  static constexpr int HE = BITS == 8 ? 1 : 4;                      // edge entries: the site byte (P16) or the whole word that holds it (P2)
  static constexpr int OFF_HALO = 2 * REGION_BYTES;                 // [2 regions][left, right][32 rows] edge entries
  static constexpr int OFF_SMETA = OFF_HALO + 128 * HE;             // SubMeta[4]
  static constexpr int STAGE_BYTES = OFF_SMETA + 128;
  static constexpr int NSTAGE = ST_DEPTH * ST_GROUPS;               // slots ST_DEPTH g .. ST_DEPTH g + ST_DEPTH - 1 belong to consumer group g
  // dynamic shared memory map (byte offsets)
  static constexpr int OFF_THR = 0;                                 // uint32 threshold[THR_STRIDE], then uint32 packed deltas[THR_STRIDE]
  static constexpr int OFF_DESC = OFF_THR + THR_STRIDE * 8;         // uint2 descriptors [8][28][16]
  static constexpr int OFF_STAGE = OFF_DESC + ST_DESC_SMEM;         // NSTAGE stage buffers
  static constexpr int OFF_BAR = OFF_STAGE + NSTAGE * STAGE_BYTES;  // full[NSTAGE], empty[NSTAGE]
  static constexpr int SMEM_BYTES = OFF_BAR + 2 * NSTAGE * 8 + 16;
};

// ---------------------------------------------------------------------------------------------------------------
// PTX helpers: mbarrier and 1-D bulk copy global -> shared (TMA engine).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// try_wait suspends the thread in hardware up to the time hint (ns): a waiter costs a handful of instructions per wake-up
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, uint32_t hint_ns) {
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity), "r"(hint_ns)
        : "memory");
  }
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// staged lattice bytes: volatile (ordered with the barrier operations); tables: plain asm, free to schedule
__device__ __forceinline__ V16 lds_v16(uint32_t addr) {
  V16 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.w[0]), "=r"(v.w[1]), "=r"(v.w[2]), "=r"(v.w[3]) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t lds_u32v(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
// staged lattice data in either tiled layout: the 16-site vector at addr, the site byte just left of a vector (the last
// site of the word / byte at addr) and just right of it (the first site of the word / byte at addr)
template <int BITS> __device__ __forceinline__ V16 lds_vec(uint32_t addr) { return BITS == 8 ? lds_v16(addr) : widen2(lds_u32v(addr)); }
template <int BITS> __device__ __forceinline__ uint32_t lds_siteL(uint32_t addr) {
  if (BITS == 8) return lds_u8(addr);
  const uint32_t w = lds_u32v(addr);
  return __funnelshift_l(w, w, 2) & 9u;       // site 15: f at bit 30, g at bit 1
}
template <int BITS> __device__ __forceinline__ uint32_t lds_siteR(uint32_t addr) { return BITS == 8 ? lds_u8(addr) : (lds_u32v(addr) & 9u); }
__device__ __forceinline__ uint2 lds_tab64(uint32_t addr) {
  uint2 v;
  asm("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t lds_tab32(uint32_t addr) {
  uint32_t v;
  asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}

// Which staged rows are read one byte to the left (bit 0) or to the right (bit 1) of the item's 16 bytes, i.e. need
// their 16-byte halo: the rows the consumers load with a shift (mirrors the shifted loads in k_staged_phase).
__device__ __forceinline__ int halo_flags(int type, int phase, int p2, int kyr, int kx) {
  if (type == PH_FAR) {
    if (kyr < 0 || kyr > 3) return 0;
    const bool arow = ((kyr ^ phase) & 1) == 0;                     // a-rows: plane 3 is the left neighbour of plane 0
    return arow ? (kx == 3 ? 1 : 0) : (kx == 0 ? 2 : 0);            // b-rows: plane 0 is the right neighbour of plane 3
  }
  if (type == PH_NEAR_V) {
    const int kya0 = (p2 + 2 * (phase & 1)) & 3, kya1 = (p2 + 2 * ((1 + phase) & 1)) & 3;
    if (kx == 3 && (kyr == kya0 || kyr == kya0 + 1)) return 1;
    if (kx == 0 && (kyr == kya1 || kyr == kya1 + 1)) return 2;
    return 0;
  }
  int f = 0;
  for (int ky = 0; ky < 4; ++ky) {                                   // horizontal dominoes of lattice row ky
    const int ka = (p2 + 2 * ((ky + phase) & 1)) & 3;
    if (ka == 3) { if ((kyr == ky && (kx == 3 || kx == 2)) || ((kyr == ky - 1 || kyr == ky + 1) && kx == 3)) f |= 1; }
    if (ka == 0 && kyr == ky && kx == 3) f |= 1;
    if (ka == 2 && kyr == ky && kx == 0) f |= 2;
  }
  return f;
}

// Philox4x32-7 (the update stream, ic_common.cuh) with the round keys precomputed on the host (PhaseArgs::rk) and the launch-constant parts of the first two
// rounds folded: counter (c0, y, c2, c3), key (k0, k1).  x0 = f0 ^ y and cb = c3 ^ rk[1] are formed once per item / block.
struct PhiloxItem { uint32_t x0, hi0, lo0; };   // x0 = c0' of round 1 (the same for the four blocks of an item), M0 * x0
__device__ __forceinline__ u32x4 philox_staged(uint32_t c0, const PhiloxItem& it, uint32_t cb, const PhaseArgs& A) {
  // round 0: (c0, y, c2, c3) -> (hi(M1 c2) ^ y ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0))
  uint32_t h, l;
  mulhilo(PHILOX_M0, c0, h, l);
  uint32_t x2 = h ^ cb, x3 = l;
  // round 1: x0 = it.x0, x1 = f1
  uint32_t h1, l1;
  mulhilo(PHILOX_M1, x2, h1, l1);
  uint32_t y0 = h1 ^ A.f2, y1 = l1, y2 = it.hi0 ^ x3 ^ A.rk[3], y3 = it.lo0;
#pragma unroll
  for (int round = 2; round < PHILOX_UPDATE_ROUNDS; ++round) {
    uint32_t a, b, c, d;
    mulhilo(PHILOX_M0, y0, a, b);
    mulhilo(PHILOX_M1, y2, c, d);
    y0 = c ^ y1 ^ A.rk[2 * round]; y1 = d; y2 = a ^ y3 ^ A.rk[2 * round + 1]; y3 = b;
  }
  u32x4 r; r.v[0] = y0; r.v[1] = y1; r.v[2] = y2; r.v[3] = y3; return r;
}

// ---------------------------------------------------------------------------------------------------------------
// Four coupled pairs (one 32-bit word of site bytes per side).  All table lookups are 4-byte shared loads: the phase
// kernels are bound by shared-memory wavefronts, and with 4-byte entries the hot entries of each table (sigma-sigma pairs,
// classes without charged neighbours) fall into distinct banks.
//   move descriptor [r][key], key = fa | fb<<1 | ga<<3 | gb<<4, r = w & 7 (the table of two-site configurations,
//   PAPER.md:66-74), 8 bytes, 16 copies so that every lane of a half warp reads its own banks (no conflicts at all):
//   coef = four int8 coefficients;  info = shared-memory address of the class base in the threshold table (low 16 bits) |
//   xor of the site bytes (a at bits 0,3; b at bits 1,4) << 16.
//   class tables [class]: threshold 8*t29 - 1 (accept iff w <= it), packed (dn2, dV, dJ).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void pairs4(uint32_t& A4, uint32_t& B4, uint32_t EA4, uint32_t EB4, uint32_t w0, uint32_t w1,
                                       uint32_t w2, uint32_t w3, uint32_t s_desc, int& a3) {
  // neighbour sums as (4F, 8G), G coefficients halved: the dp4a below yields a byte address in the 4-byte thresholds
  const uint32_t FA = (EA4 << 2) & 0x1C1C1C1Cu, GA = EA4 & 0x38383838u;
  const uint32_t FB = (EB4 << 2) & 0x1C1C1C1Cu, GB = EB4 & 0x38383838u;
  const uint32_t t0 = __byte_perm(FA, GA, 0x5140), t1 = __byte_perm(FA, GA, 0x7362);
  const uint32_t u0 = __byte_perm(FB, GB, 0x5140), u1 = __byte_perm(FB, GB, 0x7362);
  const uint32_t W0 = __byte_perm(t0, u0, 0x5410), W1 = __byte_perm(t0, u0, 0x7632);
  const uint32_t W2 = __byte_perm(t1, u1, 0x5410), W3 = __byte_perm(t1, u1, 0x7632);
  // key fa | fb<<1 | ga<<3 | gb<<4 (< 28), times 4 in each byte; a dp4a with the coefficient 32 at byte i gives key * 128,
  // the offset of the key's 16 private copies in the table [r][key][lane & 15] (address arithmetic on the FMA pipe: the
  // ALU pipe is the critical resource of this kernel)
  const uint32_t KS = 4u * A4 + 8u * B4;
  const uint2 q0 = lds_tab64((w0 & 7u) * ST_DESC_RSTRIDE + (uint32_t)__dp4a((int)KS, 0x00000020, (int)s_desc));   // s_desc includes (lane & 15) * 8
  const uint2 q1 = lds_tab64((w1 & 7u) * ST_DESC_RSTRIDE + (uint32_t)__dp4a((int)KS, 0x00002000, (int)s_desc));
  const uint2 q2 = lds_tab64((w2 & 7u) * ST_DESC_RSTRIDE + (uint32_t)__dp4a((int)KS, 0x00200000, (int)s_desc));
  const uint2 q3 = lds_tab64((w3 & 7u) * ST_DESC_RSTRIDE + (uint32_t)__dp4a((int)KS, 0x20000000, (int)s_desc));
  const uint32_t f0 = q0.x, i0 = q0.y, f1 = q1.x, i1 = q1.y, f2 = q2.x, i2 = q2.y, f3 = q3.x, i3 = q3.y;
  const uint32_t o0 = (uint32_t)__dp4a((int)W0, (int)f0, (int)(i0 & 0xFFFFu));
  const uint32_t o1 = (uint32_t)__dp4a((int)W1, (int)f1, (int)(i1 & 0xFFFFu));
  const uint32_t o2 = (uint32_t)__dp4a((int)W2, (int)f2, (int)(i2 & 0xFFFFu));
  const uint32_t o3 = (uint32_t)__dp4a((int)W3, (int)f3, (int)(i3 & 0xFFFFu));
  const uint32_t c0 = lds_tab32(o0), c1 = lds_tab32(o1), c2 = lds_tab32(o2), c3 = lds_tab32(o3);
  uint32_t D4 = 0u;
  if (w0 <= c0) { a3 += (int)lds_tab32(o0 + 4u * THR_STRIDE); D4 = __byte_perm(D4, i0, 0x3216); }
  if (w1 <= c1) { a3 += (int)lds_tab32(o1 + 4u * THR_STRIDE); D4 = __byte_perm(D4, i1, 0x3260); }
  if (w2 <= c2) { a3 += (int)lds_tab32(o2 + 4u * THR_STRIDE); D4 = __byte_perm(D4, i2, 0x3610); }
  if (w3 <= c3) { a3 += (int)lds_tab32(o3 + 4u * THR_STRIDE); D4 = __byte_perm(D4, i3, 0x6210); }
  A4 ^= D4 & 0x09090909u;
  B4 ^= (D4 >> 1) & 0x09090909u;
}
// sum over the 16 site bytes f | g<<3 of a vector: accF += sum f, accT += sum f + 8 sum g
__device__ __forceinline__ void sigma_sums(const V16& v, int& accF, int& accT) {
  const uint32_t s = v.w[0] + v.w[1] + v.w[2] + v.w[3];     // per byte: (sum f) | (sum g) << 3, both <= 4
  accT = __dp4a((int)s, 0x01010101, accT);
  accF = __dp4a((int)(s & 0x07070707u), 0x01010101, accF);
}

// store 16 bytes at plane columns X0-1 .. X0+14 of a tile row; the byte at -1 of the tile lives at `left`
__device__ __forceinline__ void st16_left1_tile(uint8_t* row, uint8_t* left, int X0, const V16& v) {
  *(X0 ? row + X0 - 1 : left) = (uint8_t)(v.w[0] & 0xFFu);
  const V16 s = shift_down(v, 0u);                       // bytes v1..v15 at X0..X0+14
  *reinterpret_cast<uint2*>(row + X0) = make_uint2(s.w[0], s.w[1]);
  *reinterpret_cast<uint32_t*>(row + X0 + 8) = s.w[2];
  *reinterpret_cast<uint16_t*>(row + X0 + 12) = (uint16_t)(s.w[3] & 0xFFFFu);
  row[X0 + 14] = (uint8_t)((s.w[3] >> 16) & 0xFFu);
}

// ---------------------------------------------------------------------------------------------------------------
// The phase kernel.  TYPE: PH_FAR / PH_NEAR_H / PH_NEAR_V; CW: word part of the FAR lane permutation.
// grid = (blocks, replicas), block = 2 groups of 256 consumer threads + 2 producer warps.
// ---------------------------------------------------------------------------------------------------------------
template <int TYPE, int CW, int BITS>
__global__ void __launch_bounds__(ST_THREADS, 1) k_staged_phase(const __grid_constant__ PhaseArgs A) {
  using C = StagedCfg<TYPE, BITS>;
  constexpr int RB = C::RB, HE = C::HE;
  constexpr int SEG = ST_SEG, LOGSEG = ST_LOGSEG, NST = C::NSTAGE;
  extern __shared__ __align__(128) unsigned char smem[];
  const int r = blockIdx.y, tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0);               // warp-uniform for the compiler
  const uint32_t smem0 = smem_u32(smem);
  const uint32_t bar0 = smem0 + C::OFF_BAR;                             // full[s] at bar0 + 8 s, empty[s] at + 8 (NST + s)
  // Programmatic dependent launch: the next kernel of the stream may start its blocks as soon as ours leave their SMs;
  // it fills its tables (which no kernel writes) and then waits for the whole of this grid before touching the lattice.
  asm volatile("griddepcontrol.launch_dependents;");
  if (tid == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(bar0 + 8 * s, 1);                                     // the producer warp (+ the bytes of its copies)
      mbar_init(bar0 + 8 * (NST + s), ST_TPG / 32);                   // the warps of the consuming group
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // From here the producers run ahead: their first bulk copies are in flight while the consumers fill the tables.

  const int lw = A.logL - 2, W = 1 << lw, Wm = W - 1;
  const int lognseg = lw - LOGSEG, nseg = 1 << lognseg;
  const int ntasks = (W << lognseg) >> 1;                               // two regions per task
  uint8_t* lat = reinterpret_cast<uint8_t*>(A.lattice) + (long long)r * A.lat_stride;
  // FAR: region rho = Y * nseg + seg pairs with rho ^ Mrho
  const int mx = A.p1, my = A.p2;
  const int Mrho = TYPE == PH_FAR ? (((my >> 2) << lognseg) | ((mx >> 2) >> LOGSEG)) : 0;
  const bool paired = TYPE == PH_FAR && Mrho != 0;
  const int hb = paired ? 31 - __clz(Mrho) : 0;
  auto region_of = [&](int t, int U) -> int {
    if (!paired) return 2 * t + U;
    const int rho0 = ((t >> hb) << (hb + 1)) | (t & ((1 << hb) - 1));
    return U ? (rho0 ^ Mrho) : rho0;
  };
  // byte offset of the tile (Y, seg) in the lattice: tiles in the order [seg][Y], 16 plane rows of SEG bytes each
  auto tile_off = [&](int Y, int seg) -> long long { return ((((long long)seg << lw) + Y) << 4) * RB; };
  // tasks of this block: t = blockIdx.x + n * gridDim.x, n = 0, 1, ...; task n belongs to consumer group g = n % ST_GROUPS
  // and is its k-th task, k = n / ST_GROUPS; it lives in slot ST_DEPTH g + k % ST_DEPTH on lap (k / ST_DEPTH) & 1.  A slot is thus always
  // drained by the same group and filled in task order, so nobody can wait on a barrier more than one phase away from
  // its own -- the only case a parity wait gets wrong.
  int tn2 = 0, tV = 0, tJ = 0, tM = 0, tMs = 0;
  int aF = 0, aT = 0, bF = 0, bT = 0, sgn = 1;   // sums over the new site bytes of the a- and b-sites (sigma_sums)

  if (warp >= ST_CONS / 32) {
    // ============================== producer warp g: both regions of every task of consumer group g =====================
    asm volatile("griddepcontrol.wait;" ::: "memory");                  // the previous phase / fold kernel is complete
    const int g = warp - ST_CONS / 32;
    const int kyr = (lane >> 2) - 1, kx = lane & 3;                     // lane = staged row (ky_rel + 1) * 4 + kx
    const int hf = lane < C::ROWS ? halo_flags(TYPE, A.phase, A.p2, kyr, kx) : 0;
    const int dY = kyr < 0 ? -1 : kyr > 3 ? 1 : 0;
    const int rowoff = (((kyr & 3) << 2) | kx) * RB;
    // the edge bytes of a task are loaded one task ahead (their latency hides behind the wait for the ring slot)
    auto halo_load = [&](int t, uint32_t (&hl)[2], uint32_t (&hr)[2]) {
      hl[0] = hl[1] = hr[0] = hr[1] = 0u;
      if (hf && t < ntasks) {
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          const int rho = region_of(t, U), Yq = rho >> lognseg, sg = rho & (nseg - 1), Yr = (Yq + dY) & Wm;
          if (BITS == 8) {
            if (hf & 1) hl[U] = lat[tile_off(Yr, (sg - 1) & (nseg - 1)) + rowoff + SEG - 1];
            if (hf & 2) hr[U] = lat[tile_off(Yr, (sg + 1) & (nseg - 1)) + rowoff];
          } else {       // the last / first word of the neighbouring tile's plane row
            if (hf & 1) hl[U] = *reinterpret_cast<const uint32_t*>(lat + tile_off(Yr, (sg - 1) & (nseg - 1)) + rowoff + RB - 4);
            if (hf & 2) hr[U] = *reinterpret_cast<const uint32_t*>(lat + tile_off(Yr, (sg + 1) & (nseg - 1)) + rowoff);
          }
        }
      }
    };
    uint32_t hl[2], hr[2];
    // The first 15/16 of the tasks are dealt statically (task b + g G + k 2G to group g of block b of G); the rest is handed
    // out by a counter of the replica in global memory (zeroed by k_fold after every sweep): whichever producer is ready
    // takes the next one, so the blocks of a launch -- and the two groups of a block -- finish within one task of each
    // other whatever the speed of their SMs (with all tasks dealt statically the SMs idle for 4 % of a launch; with all
    // tasks from the counter its one address limits the launch: about 190 atomics per microsecond).  The next task is asked
    // for one task ahead and looked at after the current stage is handed over.
    unsigned int* ctr = A.task_ctr + TASK_CTR_STRIDE * r;
    const int tstep = ST_GROUPS * (int)gridDim.x;
    const int T0 = ((ntasks - (ntasks >> 4)) / tstep) * tstep;          // static part: the same number of tasks for every producer
    int t = (int)blockIdx.x + g * (int)gridDim.x;
    if (t >= T0) {
      int tt = 0;
      if (lane == 0) tt = T0 + (int)atomicAdd(ctr, 1u);
      t = __shfl_sync(0xFFFFFFFFu, tt, 0);
    }
    halo_load(t, hl, hr);
    for (int k = 0;; ++k) {
      const int kd = k % ST_DEPTH, s = ST_DEPTH * g + kd, lap = (k / ST_DEPTH) & 1;
      const uint32_t full = bar0 + 8 * s;
      mbar_wait(bar0 + 8 * (NST + s), (uint32_t)(lap ^ 1), 20000u);
      unsigned char* stg = smem + C::OFF_STAGE + s * C::STAGE_BYTES;
      if (t >= ntasks) {
        // no task left: the group learns it from the task records (Y = -1) of one more, empty stage
        if (lane >= 28) (reinterpret_cast<SubMeta*>(stg + C::OFF_SMETA) + (lane - 28))->Y = -1;
        __syncwarp();
        if (lane == 0) mbar_arrive(full);
        break;
      }
      int Yq[2], sg[2];
#pragma unroll
      for (int U = 0; U < 2; ++U) { const int rho = region_of(t, U); Yq[U] = rho >> lognseg; sg[U] = rho & (nseg - 1); }
      if (lane == 0) {
        mbar_expect_tx(full, 2u * (uint32_t)C::REGION_BYTES);
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          const uint32_t dst = smem_u32(stg + U * C::REGION_BYTES);
          const int Y = Yq[U];
          if (Y != 0 && Y != Wm) {
            bulk_g2s(dst, lat + tile_off(Y - 1, sg[U]) + 12 * RB, C::REGION_BYTES, full);
          } else if (Y == 0) {
            bulk_g2s(dst, lat + tile_off(Wm, sg[U]) + 12 * RB, 4 * RB, full);
            bulk_g2s(dst + 4 * RB, lat + tile_off(0, sg[U]), (C::ROWS - 4) * RB, full);
          } else {
            bulk_g2s(dst, lat + tile_off(Y - 1, sg[U]) + 12 * RB, 20 * RB, full);
            bulk_g2s(dst + 20 * RB, lat + tile_off(0, sg[U]), (C::ROWS - 20) * RB, full);
          }
        }
      }
      int tn_raw = t + tstep;                            // the next task: asked for now, looked at after the stage is handed over
      if (tn_raw >= T0 && lane == 0) tn_raw = T0 + (int)atomicAdd(ctr, 1u);
      if (lane >= 28) {
        // sub-task (U, half): where its items store to, and the coordinates for the Philox counters
        const int sub = lane - 28, U = sub >> 1, half = sub & 1, Y = Yq[U], seg = sg[U];
        SubMeta mt; mt.Y = Y; mt.C0 = seg << (LOGSEG - 4); mt.pl = 0ull;
        if (TYPE == PH_FAR) {
          const int UP = paired ? (U ^ 1) : U;
          const int ky = A.phase + 2 * half, kyb = ky ^ (my & 3);
          mt.pa = (unsigned long long)(lat + tile_off(Y, seg) + (ky * 4) * RB);
          mt.pb = (unsigned long long)(lat + tile_off(Yq[UP], sg[UP]) + (kyb * 4) * RB);
        } else if (TYPE == PH_NEAR_V) {
          const int ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kyb = (ky + 1) & 3, Yb = (Y + (ky == 3)) & Wm;
          mt.pa = (unsigned long long)(lat + tile_off(Y, seg) + (ky * 4) * RB);
          mt.pb = (unsigned long long)(lat + tile_off(Yb, seg) + (kyb * 4) * RB);
        } else {
          const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
          mt.pa = (unsigned long long)(lat + tile_off(Y, seg) + (half * 4 + ka) * RB);
          mt.pb = (unsigned long long)(lat + tile_off(Y, seg) + (half * 4 + kb) * RB);
          // the last site of the same plane row of the tile to the left: its byte (P16) or the word that holds it (P2)
          mt.pl = (unsigned long long)(lat + tile_off(Y, (seg - 1) & (nseg - 1)) + (half * 4 + ka) * RB + RB - HE);
        }
        *(reinterpret_cast<SubMeta*>(stg + C::OFF_SMETA) + sub) = mt;
      }
#pragma unroll
      for (int U = 0; U < 2; ++U) {
        if (BITS == 8) {
          if (hf & 1) stg[C::OFF_HALO + U * 64 + lane] = (uint8_t)hl[U];
          if (hf & 2) stg[C::OFF_HALO + U * 64 + 32 + lane] = (uint8_t)hr[U];
        } else {
          if (hf & 1) reinterpret_cast<uint32_t*>(stg + C::OFF_HALO)[U * 64 + lane] = hl[U];
          if (hf & 2) reinterpret_cast<uint32_t*>(stg + C::OFF_HALO)[U * 64 + 32 + lane] = hr[U];
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(full);
      t = __shfl_sync(0xFFFFFFFFu, tn_raw, 0);
      halo_load(t, hl, hr);
    }
  } else {
    // =========================================== consumer warps ====================================================
    // item = one 16-byte vector of a-sites (b-sites for NEAR-H) = 16 coupled pairs: sub-task (U, half), plane/row selector
    // hi, chunk of 16 plane columns (SEG / 16 = 32 chunks = the lanes of a warp); all but the chunk are uniform in a warp
    {
      // class tables of the replica and the per-lane move descriptors of the sweep type (written by no kernel: this overlaps
      // the tail of the previous launch where two blocks fit an SM, and the producers' first copies everywhere)
      const uint2* src = A.thr + (long long)r * THR_STRIDE;
      uint32_t* thr_s = reinterpret_cast<uint32_t*>(smem + C::OFF_THR);
      const uint2* dsrc = A.desc32 + (TYPE == PH_FAR ? 0 : ST_DESC_ENTRIES);
      uint2* desc_s = reinterpret_cast<uint2*>(smem + C::OFF_DESC);
      // all loads of a thread are issued before its first store: one memory latency for the fill, not one per entry
      constexpr int NT = (THR_STRIDE + ST_CONS - 1) / ST_CONS, ND = (ST_DESC_SMEM / 8 + ST_CONS - 1) / ST_CONS;
      uint2 tv[NT], dv[ND];
#pragma unroll
      for (int i = 0; i < NT; ++i) { const int k = tid + i * ST_CONS; tv[i] = k < THR_STRIDE ? __ldg(&src[k]) : make_uint2(0u, 0u); }
#pragma unroll
      for (int i = 0; i < ND; ++i) {
        const int k = tid + i * ST_CONS, row = k >> 4, rr = row / 28, key = row - 28 * rr;   // keys with bit 2 set do not occur: null entries
        dv[i] = k < ST_DESC_SMEM / 8 ? __ldg(&dsrc[key * 8 + rr]) : make_uint2(0u, 0u);
      }
#pragma unroll
      for (int i = 0; i < NT; ++i) { const int k = tid + i * ST_CONS; if (k < THR_STRIDE) { thr_s[k] = tv[i].x; thr_s[THR_STRIDE + k] = tv[i].y; } }
#pragma unroll
      for (int i = 0; i < ND; ++i) {
        const int k = tid + i * ST_CONS;
        if (k < ST_DESC_SMEM / 8) { dv[i].y += smem0 + C::OFF_THR; desc_s[k] = dv[i]; }   // low 16 bits: shared-memory address of the class base (< 64 KB)
      }
      asm volatile("griddepcontrol.wait;" ::: "memory");                // before the first store to the lattice
      asm volatile("bar.sync 1, %0;" ::"n"(ST_CONS) : "memory");        // the consumers' tables are complete
    }
    const int g = warp >> 3, wg = warp & 7, sub = wg >> 1, hi = wg & 1, chunk = lane, U = sub >> 1, half = sub & 1, X0 = chunk << 4;
    const uint32_t s_desc = smem0 + C::OFF_DESC + (uint32_t)(lane & 15) * 8u;
    const uint32_t cb = ((uint32_t)r | (TAG_UPDATE << 28)) ^ A.rk[1];
    // byte offsets inside a stage buffer: the 16 bytes at plane column Xc of staged row (ky_rel, kx) of region UU,
    // and the bytes just left / right of them (across the tile edge: the side array filled by the producer)
    auto off = [&](int UU, int kyr, int kx, int Xc) -> int { return UU * C::REGION_BYTES + (((kyr + 1) << 2) + (kx & 3)) * RB + Xc * BITS / 8; };
    auto offL = [&](int UU, int kyr, int kx, int Xc) -> int {
      return Xc ? off(UU, kyr, kx, Xc) - HE : C::OFF_HALO + HE * (UU * 64 + ((kyr + 1) << 2) + (kx & 3));
    };
    auto offR = [&](int UU, int kyr, int kx, int Xc) -> int {
      return Xc != SEG - 16 ? off(UU, kyr, kx, Xc) + 16 * BITS / 8 : C::OFF_HALO + HE * (UU * 64 + 32 + ((kyr + 1) << 2) + (kx & 3));
    };
    // ---- thread-constant offsets of everything the item loads (relative to the stage buffer) --------------------------
    // o[0] a, o[1] b, o[2..] neighbour vectors; h[..] bytes across the vector's edge for the shifted loads
    int oa, ob, on[4], oh[4], kxr, ky_ctr;
    int sh_a = 0, sh_l = 0, sh_r = 0;
    uint32_t selb = 0x3210u;
    int goffa, goffb;                          // byte offsets of the item's stores from SubMeta::pa / pb
    bool left1 = false;
    if (TYPE == PH_FAR) {
      const int ky = A.phase + 2 * half, kxa = 2 * hi;
      const int kyb = ky ^ (my & 3), UB = paired ? (U ^ 1) : U, kxb = kxa ^ (mx & 3);
      const int Xb = X0 ^ ((mx >> 2) & (SEG - 1) & ~15);               // the partner chunk inside the partner tile
      sgn = A.phase ? -1 : 1;
      oa = off(U, ky, kxa, X0); ob = off(UB, kyb, kxb, Xb);
      on[0] = off(U, ky, kxa + 3, X0); on[1] = off(U, ky, kxa + 1, X0);          // left (shifted if kxa == 0), right of a
      on[2] = off(UB, kyb, kxb + 3, Xb); on[3] = off(UB, kyb, kxb + 1, Xb);      // left, right (shifted if kxb == 3) of b
      oh[0] = offL(U, ky, kxa + 3, X0); oh[1] = offR(UB, kyb, kxb + 1, Xb); oh[2] = oh[3] = 0;
      sh_l = kxa == 0; sh_r = kxb == 3;
      selb = 0x3210u ^ (0x1111u * (uint32_t)((mx >> 2) & 3));          // byte part of the lane permutation i -> i ^ (mx >> 2 & 15)
      ky_ctr = ky; kxr = kxa;
      goffa = (kxa * SEG + X0) * BITS / 8; goffb = (kxb * SEG + Xb) * BITS / 8;
    } else if (TYPE == PH_NEAR_V) {
      const int kx = half + 2 * hi, ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3;
      sgn = ((half + ky) & 1) ? -1 : 1;
      oa = off(U, ky, kx, X0); ob = off(U, ky + 1, kx, X0);            // row 4 = row 0 of the quad below
      on[0] = off(U, ky, kx + 3, X0); on[1] = off(U, ky, kx + 1, X0);
      on[2] = off(U, ky + 1, kx + 3, X0); on[3] = off(U, ky + 1, kx + 1, X0);
      sh_l = kx == 0; sh_r = kx == 3;
      oh[0] = sh_l ? offL(U, ky, kx + 3, X0) : offR(U, ky, kx + 1, X0);
      oh[1] = sh_l ? offL(U, ky + 1, kx + 3, X0) : offR(U, ky + 1, kx + 1, X0);
      oh[2] = oh[3] = 0;
      ky_ctr = ky; kxr = kx;
      goffa = (kx * SEG + X0) * BITS / 8; goffb = goffa;
    } else {
      // NEAR, horizontal dominoes of row ky = half + 2 hi; lanes are indexed by the b-site
      const int ky = half + 2 * hi;
      const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
      sh_a = ka == 3; sh_l = sh_a || ka == 0; sh_r = kb == 3;
      sgn = ((ka + half) & 1) ? -1 : 1;
      oa = off(U, ky, ka, X0); ob = off(U, ky, kb, X0);
      on[0] = off(U, ky, ka + 3, X0); on[1] = off(U, ky, kb + 1, X0);            // left of a, right of b
      on[2] = 0; on[3] = 0;
      oh[0] = offL(U, ky, ka, X0);                                               // a, a-up, a-down: +- 4 rows from here
      oh[1] = offL(U, ky, ka + 3, X0); oh[2] = offR(U, ky, kb + 1, X0); oh[3] = 0;
      ky_ctr = ky; kxr = kb;
      left1 = sh_a != 0;
      goffa = 8 * hi * RB; goffb = 8 * hi * RB + X0 * BITS / 8;        // plane rows (ky, ka), (ky, kb)
    }
    constexpr int ROW4 = 4 * RB;                                       // four staged rows = one lattice row up / down
    const uint32_t stg_g = smem0 + C::OFF_STAGE + ST_DEPTH * g * C::STAGE_BYTES;
    const SubMeta* meta_g = reinterpret_cast<const SubMeta*>(smem + C::OFF_STAGE + ST_DEPTH * g * C::STAGE_BYTES + C::OFF_SMETA) + sub;

    for (int k = 0;; ++k) {
      const int kd = k % ST_DEPTH, s = ST_DEPTH * g + kd, lap = (k / ST_DEPTH) & 1;
      const uint32_t st = stg_g + kd * C::STAGE_BYTES;
      mbar_wait(bar0 + 8 * s, (uint32_t)lap, 1000u);
      const SubMeta* mp = reinterpret_cast<const SubMeta*>(reinterpret_cast<const unsigned char*>(meta_g) + kd * C::STAGE_BYTES);
      const int Y = mp->Y, chunkG = mp->C0 + chunk;
      if (Y < 0) break;                                                 // the producer found no task left
      uint8_t* gpa = reinterpret_cast<uint8_t*>(mp->pa) + goffa;
      uint8_t* gpb = reinterpret_cast<uint8_t*>(mp->pb) + goffb;
      uint8_t* gpl = nullptr;
      V16 a, b, ea, eb;
      if (TYPE == PH_FAR) {
        a = lds_vec<BITS>(st + oa); b = lds_vec<BITS>(st + ob);
        V16 l = lds_vec<BITS>(st + on[0]);
        if (sh_l) l = shift_up(l, lds_siteL<BITS>(st + oh[0]));
        ea = add(add(l, lds_vec<BITS>(st + on[1])), add(lds_vec<BITS>(st + oa - ROW4), lds_vec<BITS>(st + oa + ROW4)));
        V16 rr = lds_vec<BITS>(st + on[3]);
        if (sh_r) rr = shift_down(rr, lds_siteR<BITS>(st + oh[1]));
        eb = add(add(lds_vec<BITS>(st + on[2]), rr), add(lds_vec<BITS>(st + ob - ROW4), lds_vec<BITS>(st + ob + ROW4)));
        b = xor_perm<CW>(b, selb); eb = xor_perm<CW>(eb, selb);          // b into a's lane order (lane i <-> i ^ c)
      } else if (TYPE == PH_NEAR_V) {
        a = lds_vec<BITS>(st + oa); b = lds_vec<BITS>(st + ob);
        V16 al = lds_vec<BITS>(st + on[0]), ar = lds_vec<BITS>(st + on[1]), bl = lds_vec<BITS>(st + on[2]), br = lds_vec<BITS>(st + on[3]);
        if (sh_l) { al = shift_up(al, lds_siteL<BITS>(st + oh[0])); bl = shift_up(bl, lds_siteL<BITS>(st + oh[1])); }
        if (sh_r) { ar = shift_down(ar, lds_siteR<BITS>(st + oh[0])); br = shift_down(br, lds_siteR<BITS>(st + oh[1])); }
        // vertical domino: a's lower neighbour is b, b's upper neighbour is a
        ea = add(add(al, ar), add(lds_vec<BITS>(st + oa - ROW4), b));
        eb = add(add(bl, br), add(a, lds_vec<BITS>(st + ob + ROW4)));
      } else {
        a = lds_vec<BITS>(st + oa); b = lds_vec<BITS>(st + ob);
        V16 au = lds_vec<BITS>(st + oa - ROW4), ad = lds_vec<BITS>(st + oa + ROW4), al = lds_vec<BITS>(st + on[0]), br = lds_vec<BITS>(st + on[1]);
        if (sh_a) {
          a = shift_up(a, lds_siteL<BITS>(st + oh[0]));
          au = shift_up(au, lds_siteL<BITS>(st + oh[0] + (X0 ? -ROW4 : -4 * HE))); ad = shift_up(ad, lds_siteL<BITS>(st + oh[0] + (X0 ? ROW4 : 4 * HE)));
        }
        if (sh_l) al = shift_up(al, lds_siteL<BITS>(st + oh[1]));
        if (sh_r) br = shift_down(br, lds_siteR<BITS>(st + oh[2]));
        ea = add(add(al, b), add(au, ad));
        eb = add(add(a, br), add(lds_vec<BITS>(st + ob - ROW4), lds_vec<BITS>(st + ob + ROW4)));
        gpl = reinterpret_cast<uint8_t*>(mp->pl) + goffa;
      }
      V16 a_old;
      if (BITS == 2 && TYPE == PH_NEAR_H) a_old = a;
      // everything the item needs is in registers: hand the ring slot back to the producers before the long part
      __syncwarp();
      if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s));
      // random words: block c0 = 4*(X>>2) + kx, c1 = y, word X & 3 of the slot site (U3)
      PhiloxItem it;
      it.x0 = A.f0 ^ (uint32_t)(4 * Y + ky_ctr);
      mulhilo(PHILOX_M0, it.x0, it.hi0, it.lo0);
      const uint32_t c0base = (uint32_t)(16 * chunkG + kxr);
      int a3 = 0;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const u32x4 rr = philox_staged(c0base + 4u * j, it, cb, A);
        pairs4(a.w[j], b.w[j], ea.w[j], eb.w[j], rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, a3);
      }
      if (TYPE == PH_FAR) b = xor_perm<CW>(b, selb);
      sigma_sums(a, aF, aT); sigma_sums(b, bF, bT);
      if (BITS == 8) {
        st16(gpb, b);
        if (TYPE == PH_NEAR_H) { if (!left1) st16(gpa + X0, a); else st16_left1_tile(gpa, gpl, X0, a); }
        else st16(gpa, a);
      } else {
        *reinterpret_cast<uint32_t*>(gpb) = pack2(b);
        if (TYPE == PH_NEAR_H && left1) {
          // the vector holds the sites X0-1 .. X0+14: site X0-1 lives in the word to the left (owned by the neighbouring
          // lane, or by another block across the tile edge) and site X0+15 of this word is somebody else's, so the
          // changes are xor-ed in (commutative: no order between the two writers of a word is needed)
          const V16 d = {{a.w[0] ^ a_old.w[0], a.w[1] ^ a_old.w[1], a.w[2] ^ a_old.w[2], a.w[3] ^ a_old.w[3]}};
          const uint32_t own = pack2(shift_down(d, 0u)), prev = __funnelshift_l(d.w[0] & 9u, d.w[0] & 9u, 30);
          uint32_t* wa = reinterpret_cast<uint32_t*>(gpa) + chunk;
          if (own) atomicXor(wa, own);
          if (prev) atomicXor(X0 ? wa - 1 : reinterpret_cast<uint32_t*>(gpl), prev);
        } else {
          *reinterpret_cast<uint32_t*>(TYPE == PH_NEAR_H ? gpa + X0 / 4 : gpa) = pack2(a);
        }
      }
      // unpack the item's sums: a3 = dJ + (dV << 11) + (dn2 << 22)
      const int j11 = (a3 << 21) >> 21; a3 = (a3 - j11) >> 11;
      const int v11 = (a3 << 21) >> 21; a3 = (a3 - v11) >> 11;
      tJ += j11; tV += v11; tn2 += a3;
    }
    // M and Ms of the sites this thread updated, from their new values: sum sigma = sum f - sum g = (9 accF - accT) / 8.
    // Every site is active in exactly one phase of a sweep, so the two phases add up to the whole lattice (k_fold).
    const int Ma = (9 * aF - aT) >> 3, Mb = (9 * bF - bT) >> 3;
    tM = Ma + Mb;
    tMs = sgn * (TYPE == PH_FAR ? Ma + Mb : Ma - Mb);      // FAR: all active sites have one colour; NEAR: a and b differ
  }
  block_accumulate(&A.obs[r], tn2, tV, tJ, tM, tMs, true);
}

}  // namespace ic
