// ic_kernels_staged.cuh -- variant 3: the production sm_100a kernels for L >= 2048 on the tiled layout LAY_P16.
//
// One launch = one phase of a sweep (schedule S1, U4), one persistent block per SM:
//   * 4 producer warps stage "regions" of the lattice in shared memory with 1-D bulk copies (cp.async.bulk, the TMA
//     engine; completion on an mbarrier).  A region is one tile of the layout (row quad Y, 512 plane columns: 16 plane
//     rows = 8 KB contiguous in global memory, ONE copy) plus the plane rows of the lattice row above and of the one
//     (NEAR-V: two) below (2 KB / 4 KB contiguous, one copy each).  The few bytes read across the left/right tile
//     edge (the x-1 neighbour of plane 0 is plane 3 one byte to the left) are fetched by the producer's other lanes
//     with plain loads into a small side array.  Bulk copies cost ~120 cycles of issue each whatever their size
//     (measured), which is why the layout makes a region three copies and not twenty.
//   * 16 consumer warps in 4 groups; group g processes tasks g, g+4, ... of the block, task n lives in ring slot
//     n mod NSTAGE.  A task is two regions = 4096 coupled pairs.  In a FAR phase the two regions are partners under
//     (x^mx, y^my): every byte of both is loaded once and all pairs between them are updated.
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

constexpr int ST_GROUPS = 4;                  // consumer groups per block
constexpr int ST_NPROD = 4;                   // producer warps per block
constexpr int ST_LOGSEG = P16_LOGSEG_MAX, ST_SEG = 1 << ST_LOGSEG;   // plane columns per region = per tile of the layout
constexpr int ST_TPG = ST_SEG / 4;            // consumer threads per group: one 32-pair item each per task
constexpr int ST_THREADS = 32 * ST_NPROD + ST_GROUPS * ST_TPG;
constexpr int ST_DESC_ENTRIES = 256;          // move descriptors [key*8 + r] (224 used) as two 4-byte tables: coefficients, info

template <int TYPE>
struct StagedCfg {
  static constexpr int ROWS = TYPE == PH_NEAR_V ? 28 : 24;          // staged plane rows: (ky_rel + 1) * 4 + kx, ky_rel = -1..4 (5)
  static constexpr int REGION_BYTES = ROWS * ST_SEG;
  static constexpr int OFF_HALO = 2 * REGION_BYTES;                 // uint8 [2 regions][left, right][32 rows]
  static constexpr int OFF_SMETA = OFF_HALO + 128;                  // SubMeta[4]
  static constexpr int STAGE_BYTES = OFF_SMETA + 256;
  static constexpr int NSTAGE = TYPE == PH_NEAR_V ? 6 : 7;
  static constexpr int TASK_TX = 2 * (16 + 4 + (ROWS - 20)) * ST_SEG;   // bytes the bulk copies of one task deliver
  // dynamic shared memory map (byte offsets)
  static constexpr int OFF_THR = 0;                                 // uint32 threshold[THR_STRIDE], then uint32 packed deltas[THR_STRIDE]
  static constexpr int OFF_DESC = OFF_THR + THR_STRIDE * 8;         // uint32 coef[256], then uint32 info[256]
  static constexpr int OFF_STAGE = OFF_DESC + ST_DESC_ENTRIES * 8;  // NSTAGE stage buffers
  static constexpr int OFF_BAR = OFF_STAGE + NSTAGE * STAGE_BYTES;  // full[NSTAGE], empty[NSTAGE]
  static constexpr int SMEM_BYTES = OFF_BAR + 2 * NSTAGE * 8 + 16;
};

// What the consumers of one sub-task (region U, half) need to know about the task in a stage.
struct SubMeta {
  unsigned long long pa;     // global address of the a-side plane row (see the consumers)
  unsigned long long pb;     // global address of the b-side plane row
  unsigned long long pl;     // NEAR-H: address of the byte left of the a-side plane row (last byte of the tile to the left)
  int Y, S0;                 // row quad and first plane column of the sub-task's region (Philox counters)
  int pad[8];
};
static_assert(sizeof(SubMeta) == 64, "SubMeta layout");

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
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  while (!ok) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// read-only tables in shared memory: plain (non-volatile) asm so that the compiler may schedule them freely
__device__ __forceinline__ uint4 lds_tab128(uint32_t addr) {
  uint4 v;
  asm("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint2 lds_tab64(uint32_t addr) {
  uint2 v;
  asm("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
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

// ---------------------------------------------------------------------------------------------------------------
// Four coupled pairs (one 32-bit word of site bytes per side).  All table lookups are 4-byte shared loads: the phase
// kernels are bound by shared-memory wavefronts, and with 4-byte entries the hot entries of each table (sigma-sigma pairs,
// classes without charged neighbours) fall into distinct banks.
//   move descriptor [key*8 + r], key = fa | fb<<1 | ga<<3 | gb<<4, r = w & 7 (the table of two-site configurations,
//   PAPER.md:66-74):  coef = four int8 coefficients;  info = byte offset of the class base in the threshold table (low 16
//   bits) | xor of the site bytes (a at bits 0,3; b at bits 1,4) << 16.
//   class tables [class]: threshold 8*t29 - 1 (accept iff w <= it), packed (dn2, dV, dJ).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lds_tab32(uint32_t addr) {
  uint32_t v;
  asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void pairs4(uint32_t& A4, uint32_t& B4, uint32_t EA4, uint32_t EB4, uint32_t w0, uint32_t w1,
                                       uint32_t w2, uint32_t w3, uint32_t s_desc, uint32_t s_thr, int& a3) {
  // neighbour sums scaled by 4: the dp4a below yields a byte offset into the table of 4-byte thresholds
  const uint32_t FA = (EA4 << 2) & 0x1C1C1C1Cu, GA = (EA4 >> 1) & 0x1C1C1C1Cu;
  const uint32_t FB = (EB4 << 2) & 0x1C1C1C1Cu, GB = (EB4 >> 1) & 0x1C1C1C1Cu;
  const uint32_t t0 = __byte_perm(FA, GA, 0x5140), t1 = __byte_perm(FA, GA, 0x7362);
  const uint32_t u0 = __byte_perm(FB, GB, 0x5140), u1 = __byte_perm(FB, GB, 0x7362);
  const uint32_t W0 = __byte_perm(t0, u0, 0x5410), W1 = __byte_perm(t0, u0, 0x7632);
  const uint32_t W2 = __byte_perm(t1, u1, 0x5410), W3 = __byte_perm(t1, u1, 0x7632);
  const uint32_t KEY8 = (A4 + 2u * B4) << 3;              // per byte: 8 * key  (key < 28)
  const uint32_t e0 = s_desc + 4u * (__byte_perm(KEY8, 0u, 0x4440) | (w0 & 7u));
  const uint32_t e1 = s_desc + 4u * (__byte_perm(KEY8, 0u, 0x4441) | (w1 & 7u));
  const uint32_t e2 = s_desc + 4u * (__byte_perm(KEY8, 0u, 0x4442) | (w2 & 7u));
  const uint32_t e3 = s_desc + 4u * (__byte_perm(KEY8, 0u, 0x4443) | (w3 & 7u));
  const uint32_t f0 = lds_tab32(e0), i0 = lds_tab32(e0 + 4u * ST_DESC_ENTRIES);
  const uint32_t f1 = lds_tab32(e1), i1 = lds_tab32(e1 + 4u * ST_DESC_ENTRIES);
  const uint32_t f2 = lds_tab32(e2), i2 = lds_tab32(e2 + 4u * ST_DESC_ENTRIES);
  const uint32_t f3 = lds_tab32(e3), i3 = lds_tab32(e3 + 4u * ST_DESC_ENTRIES);
  const uint32_t o0 = s_thr + (uint32_t)__dp4a((int)W0, (int)f0, (int)(i0 & 0xFFFFu));
  const uint32_t o1 = s_thr + (uint32_t)__dp4a((int)W1, (int)f1, (int)(i1 & 0xFFFFu));
  const uint32_t o2 = s_thr + (uint32_t)__dp4a((int)W2, (int)f2, (int)(i2 & 0xFFFFu));
  const uint32_t o3 = s_thr + (uint32_t)__dp4a((int)W3, (int)f3, (int)(i3 & 0xFFFFu));
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

// neighbour sums in x of the two vectors (planes sel, sel+2) of one lattice row; r0 = the 16 bytes of the plane between
// them, r1 = of the plane on the other side, e = the byte of r1 just left (sel = 0) / right (sel = 1) of them
__device__ __forceinline__ void xnbr_sums_s(const uint8_t* r0, const uint8_t* r1, const uint8_t* e, int sel, V16& s_lo, V16& s_hi) {
  const V16 q0 = ld16(r0), q1 = ld16(r1);
  if (sel == 0) { s_lo = add(q0, shift_up(q1, *e)); s_hi = add(q0, q1); }
  else { s_lo = add(q0, q1); s_hi = add(q0, shift_down(q1, *e)); }
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
// grid = (blocks, replicas), block = 4 producer warps + 4 groups of 128 consumer threads.
// ---------------------------------------------------------------------------------------------------------------
template <int TYPE, int CW>
__global__ void __launch_bounds__(ST_THREADS, 1) k_staged_phase(PhaseArgs A) {
  using C = StagedCfg<TYPE>;
  constexpr int SEG = ST_SEG, LOGSEG = ST_LOGSEG, NST = C::NSTAGE;
  extern __shared__ __align__(128) unsigned char smem[];
  const int r = blockIdx.y, tid = threadIdx.x, lane = tid & 31;
  const uint32_t bar0 = smem_u32(smem + C::OFF_BAR);                    // full[s] at bar0 + 8 s, empty[s] at + 8 (NST + s)
  {
    const uint2* src = A.thr + (long long)r * THR_STRIDE;
    uint32_t* thr_s = reinterpret_cast<uint32_t*>(smem + C::OFF_THR);
    for (int k = tid; k < THR_STRIDE; k += ST_THREADS) { const uint2 v = __ldg(&src[k]); thr_s[k] = v.x; thr_s[THR_STRIDE + k] = v.y; }
    const uint2* dsrc = A.desc32 + (TYPE == PH_FAR ? 0 : ST_DESC_ENTRIES);
    uint32_t* desc_s = reinterpret_cast<uint32_t*>(smem + C::OFF_DESC);
    for (int k = tid; k < ST_DESC_ENTRIES; k += ST_THREADS) { const uint2 v = __ldg(&dsrc[k]); desc_s[k] = v.x; desc_s[ST_DESC_ENTRIES + k] = v.y; }
    if (tid == 0) {
      for (int s = 0; s < NST; ++s) {
        mbar_init(bar0 + 8 * s, 2);                                     // producer lane 0: expect_tx, and after the edge bytes
        mbar_init(bar0 + 8 * (NST + s), ST_TPG / 32);                   // the warps of the consuming group
      }
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
  }
  __syncthreads();

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
  // tasks of this block: t = blockIdx.x + n * gridDim.x, n = 0, 1, ...; task n uses ring slot n % NST
  int tn2 = 0, tV = 0, tJ = 0, tM = 0, tMs = 0;
  int aF = 0, aT = 0, bF = 0, bT = 0, sgn = 1;   // sums over the new site bytes of the a- and b-sites (sigma_sums)

  if (tid < 32 * ST_NPROD) {
    // ============================== producer warps: warp p fills the ring slots s with s % ST_NPROD == p ================
    const int p = tid >> 5;
    const int hf = lane < C::ROWS ? halo_flags(TYPE, A.phase, A.p2, (lane >> 2) - 1, lane & 3) : 0;   // lane = staged row
    // a ring slot is always filled by the same producer warp (slot % ST_NPROD), in task order: a parity wait is only
    // safe for a waiter that is at most one phase ahead of the barrier
    for (int n = 0, t = blockIdx.x; t < ntasks; ++n, t += gridDim.x) {
      const int s = n % NST;
      if (s % ST_NPROD != p) continue;
      mbar_wait(bar0 + 8 * (NST + s), ((n / NST) & 1) ^ 1);
      unsigned char* stg = smem + C::OFF_STAGE + s * C::STAGE_BYTES;
      const uint32_t full = bar0 + 8 * s;
      int Yq[2], sg[2];
#pragma unroll
      for (int U = 0; U < 2; ++U) { const int rho = region_of(t, U); Yq[U] = rho >> lognseg; sg[U] = rho & (nseg - 1); }
      if (lane == 0) {
        mbar_arrive_expect_tx(full, (uint32_t)C::TASK_TX);
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          const uint32_t dst = smem_u32(stg + U * C::REGION_BYTES);
          bulk_g2s(dst + 4 * SEG, lat + p16_row(lw, 0, 0, Yq[U], sg[U]), 16 * SEG, full);
          bulk_g2s(dst, lat + p16_row(lw, 3, 0, (Yq[U] - 1) & Wm, sg[U]), 4 * SEG, full);
          bulk_g2s(dst + 20 * SEG, lat + p16_row(lw, 0, 0, (Yq[U] + 1) & Wm, sg[U]), (C::ROWS - 20) * SEG, full);
        }
        for (int sub = 0; sub < 4; ++sub) {
          // sub-task (U, half): where its items store to, and the coordinates for the Philox counters
          const int U = sub >> 1, half = sub & 1, Y = Yq[U], seg = sg[U];
          SubMeta mt; mt.Y = Y; mt.S0 = seg << LOGSEG; mt.pl = 0ull;
          if (TYPE == PH_FAR) {
            const int UP = paired ? (U ^ 1) : U;
            const int ky = A.phase + 2 * half, kyb = ky ^ (my & 3);
            mt.pa = (unsigned long long)(lat + p16_row(lw, ky, 0, Y, seg));
            mt.pb = (unsigned long long)(lat + p16_row(lw, kyb, mx & 3, Yq[UP], sg[UP]));
          } else if (TYPE == PH_NEAR_V) {
            const int ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kyb = (ky + 1) & 3, Yb = (Y + (ky == 3)) & Wm;
            mt.pa = (unsigned long long)(lat + p16_row(lw, ky, half, Y, seg));
            mt.pb = (unsigned long long)(lat + p16_row(lw, kyb, half, Yb, seg));
          } else {
            const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
            mt.pa = (unsigned long long)(lat + p16_row(lw, half, ka, Y, seg));
            mt.pb = (unsigned long long)(lat + p16_row(lw, half, kb, Y, seg));
            mt.pl = (unsigned long long)(lat + p16_row(lw, half, ka, Y, (seg - 1) & (nseg - 1)) + SEG - 1);
          }
          reinterpret_cast<SubMeta*>(stg + C::OFF_SMETA)[sub] = mt;
        }
      }
      if (hf) {
        // bytes across the tile edge: lane = staged row (ky_rel + 1) * 4 + kx
        const int kyr = (lane >> 2) - 1, kx = lane & 3, ky = kyr & 3;
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          const int Yr = kyr < 0 ? ((Yq[U] - 1) & Wm) : kyr > 3 ? ((Yq[U] + 1) & Wm) : Yq[U];
          if (hf & 1) stg[C::OFF_HALO + U * 64 + lane] = lat[p16_row(lw, ky, kx, Yr, (sg[U] - 1) & (nseg - 1)) + SEG - 1];
          if (hf & 2) stg[C::OFF_HALO + U * 64 + 32 + lane] = lat[p16_row(lw, ky, kx, Yr, (sg[U] + 1) & (nseg - 1))];
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(full);
    }
  } else {
    // =========================================== consumer warps ====================================================
    const int ct = tid - 32 * ST_NPROD, g = ct / ST_TPG, tg = ct - g * ST_TPG;
    const int sub = tg >> 5, chunk = tg & 31, U = sub >> 1, half = sub & 1, X0 = chunk << 4;   // SEG / 16 = 32 chunks
    const uint32_t s_thr = smem_u32(smem + C::OFF_THR);
    const uint32_t s_desc = smem_u32(smem + C::OFF_DESC);
    const uint32_t c3 = (uint32_t)r | (TAG_UPDATE << 28);
    // byte offsets inside a stage buffer: the 16 bytes at plane column Xc of staged row (ky_rel, kx) of region UU,
    // and the bytes just left / right of them (across the tile edge: the side array filled by the producer)
    auto off = [&](int UU, int kyr, int kx, int Xc) -> int { return UU * C::REGION_BYTES + ((((kyr + 1) << 2) + (kx & 3)) << LOGSEG) + Xc; };
    auto offL = [&](int UU, int kyr, int kx, int Xc) -> int {
      return Xc ? off(UU, kyr, kx, Xc) - 1 : C::OFF_HALO + UU * 64 + ((kyr + 1) << 2) + (kx & 3);
    };
    auto offR = [&](int UU, int kyr, int kx, int Xc) -> int {
      return Xc != SEG - 16 ? off(UU, kyr, kx, Xc) + 16 : C::OFF_HALO + UU * 64 + 32 + ((kyr + 1) << 2) + (kx & 3);
    };
    for (int n = g, t = blockIdx.x + g * gridDim.x; t < ntasks; n += ST_GROUPS, t += ST_GROUPS * gridDim.x) {
      const int s = n % NST;
      mbar_wait(bar0 + 8 * s, (n / NST) & 1);
      const uint8_t* st = smem + C::OFF_STAGE + s * C::STAGE_BYTES;
      const SubMeta* mp = reinterpret_cast<const SubMeta*>(st + C::OFF_SMETA) + sub;
      const int Y = mp->Y, chunkG = (mp->S0 >> 4) + chunk;
      uint8_t* const gpa = reinterpret_cast<uint8_t*>(mp->pa);
      uint8_t* const gpb = reinterpret_cast<uint8_t*>(mp->pb);
      int a3 = 0;

      if (TYPE == PH_FAR || TYPE == PH_NEAR_V) {
        int sel, ky, kyb_r, UB, kxb_lo, kxb_hi, Xb = X0;
        uint32_t selb = 0x3210u;
        if (TYPE == PH_FAR) {
          sel = 0; ky = A.phase + 2 * half;
          kyb_r = ky ^ (my & 3); UB = paired ? (U ^ 1) : U;
          kxb_lo = mx & 3; kxb_hi = 2 ^ (mx & 3);
          Xb = X0 ^ ((mx >> 2) & (SEG - 1) & ~15);                     // the partner chunk inside the partner tile
          const int cb = (mx >> 2) & 3;
          selb = cb == 0 ? 0x3210u : cb == 1 ? 0x2301u : cb == 2 ? 0x1032u : 0x0123u;
          sgn = A.phase ? -1 : 1;
        } else {
          sel = half; ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3;
          kyb_r = ky + 1; UB = U;                                        // may be row 4 = row 0 of the quad below
          kxb_lo = sel; kxb_hi = sel + 2;
          sgn = ((sel + ky) & 1) ? -1 : 1;
        }
        const int y = 4 * Y + ky;
        // a side: planes (sel, sel+2); x-neighbours are planes sel+1 and sel+3 (one byte to the left / right when wrapping)
        V16 a_lo = ld16(st + off(U, ky, sel, X0)), a_hi = ld16(st + off(U, ky, sel + 2, X0));
        V16 ea_lo, ea_hi;
        xnbr_sums_s(st + off(U, ky, sel + 1, X0), st + off(U, ky, sel + 3, X0),
                    st + (sel == 0 ? offL(U, ky, sel + 3, X0) : offR(U, ky, sel + 3, X0)), sel, ea_lo, ea_hi);
        ea_lo = add(ea_lo, ld16(st + off(U, ky - 1, sel, X0)));
        ea_hi = add(ea_hi, ld16(st + off(U, ky - 1, sel + 2, X0)));
        // b side, natural lane order
        const int selp = TYPE == PH_FAR ? 1 : sel;          // b-planes are (selp, selp + 2)
        V16 b_lo = ld16(st + off(UB, kyb_r, kxb_lo, Xb)), b_hi = ld16(st + off(UB, kyb_r, kxb_hi, Xb));
        V16 eb_lo, eb_hi;
        {
          V16 s_first, s_second;
          xnbr_sums_s(st + off(UB, kyb_r, selp + 1, Xb), st + off(UB, kyb_r, selp + 3, Xb),
                      st + (selp == 0 ? offL(UB, kyb_r, selp + 3, Xb) : offR(UB, kyb_r, selp + 3, Xb)), selp, s_first, s_second);
          if (TYPE == PH_FAR) { const bool sw = (kxb_lo == 3); eb_lo = sw ? s_second : s_first; eb_hi = sw ? s_first : s_second; }
          else { eb_lo = s_first; eb_hi = s_second; }
          eb_lo = add(eb_lo, ld16(st + off(UB, kyb_r + 1, kxb_lo, Xb)));
          eb_hi = add(eb_hi, ld16(st + off(UB, kyb_r + 1, kxb_hi, Xb)));
        }
        if (TYPE == PH_FAR) {
          ea_lo = add(ea_lo, ld16(st + off(U, ky + 1, 0, X0)));
          ea_hi = add(ea_hi, ld16(st + off(U, ky + 1, 2, X0)));
          eb_lo = add(eb_lo, ld16(st + off(UB, kyb_r - 1, kxb_lo, Xb)));
          eb_hi = add(eb_hi, ld16(st + off(UB, kyb_r - 1, kxb_hi, Xb)));
          b_lo = xor_perm<CW>(b_lo, selb); b_hi = xor_perm<CW>(b_hi, selb);
          eb_lo = xor_perm<CW>(eb_lo, selb); eb_hi = xor_perm<CW>(eb_hi, selb);
        } else {
          // vertical domino: a's lower neighbour is b, b's upper neighbour is a
          ea_lo = add(ea_lo, b_lo); ea_hi = add(ea_hi, b_hi);
          eb_lo = add(eb_lo, a_lo); eb_hi = add(eb_hi, a_hi);
        }
        // random words: block (c0 = x>>3, c1 = y), word (x>>1)&3  (U3)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const u32x4 r0 = philox4x32_10((uint32_t)(8 * chunkG + 2 * j), (uint32_t)y, A.c2, c3, A.key0, A.key1);
          const u32x4 r1 = philox4x32_10((uint32_t)(8 * chunkG + 2 * j + 1), (uint32_t)y, A.c2, c3, A.key0, A.key1);
          pairs4(a_lo.w[j], b_lo.w[j], ea_lo.w[j], eb_lo.w[j], r0.v[0], r0.v[2], r1.v[0], r1.v[2], s_desc, s_thr, a3);
          pairs4(a_hi.w[j], b_hi.w[j], ea_hi.w[j], eb_hi.w[j], r0.v[1], r0.v[3], r1.v[1], r1.v[3], s_desc, s_thr, a3);
        }
        if (TYPE == PH_FAR) { b_lo = xor_perm<CW>(b_lo, selb); b_hi = xor_perm<CW>(b_hi, selb); }
        sigma_sums(a_lo, aF, aT); sigma_sums(a_hi, aF, aT); sigma_sums(b_lo, bF, bT); sigma_sums(b_hi, bF, bT);
        st16(gpa + X0, a_lo); st16(gpa + 2 * SEG + X0, a_hi);
        st16(gpb + Xb, b_lo); st16(gpb + (kxb_hi - kxb_lo) * SEG + Xb, b_hi);
      } else {
        // ---- NEAR, horizontal dominoes: rows ky = half and half + 2 share ka; lanes are indexed by the b-site ----------
        const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
        const int sh_a = -(ka == 3), sh_l = sh_a - (ka == 0), sh_r = (kb == 3);
        sgn = ((ka + half) & 1) ? -1 : 1;
        auto ldrow = [&](int kyr, int kx, int sh) -> V16 {
          V16 v = ld16(st + off(U, kyr, kx, X0));
          if (sh < 0) v = shift_up(v, st[offL(U, kyr, kx, X0)]);
          else if (sh > 0) v = shift_down(v, st[offR(U, kyr, kx, X0)]);
          return v;
        };
#pragma unroll
        for (int v = 0; v < 2; ++v) {
          const int ky = half + 2 * v, y = 4 * Y + ky;
          V16 a = ldrow(ky, ka, sh_a), b = ld16(st + off(U, ky, kb, X0));
          V16 ea = add(add(ldrow(ky, ka + 3, sh_l), b), add(ldrow(ky - 1, ka, sh_a), ldrow(ky + 1, ka, sh_a)));
          V16 eb = add(add(a, ldrow(ky, kb + 1, sh_r)), add(ld16(st + off(U, ky - 1, kb, X0)), ld16(st + off(U, ky + 1, kb, X0))));
          // random words: block (c0 = xb>>4, c1 = y), word (xb>>2)&3
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const u32x4 rr = philox4x32_10((uint32_t)(4 * chunkG + j), (uint32_t)y, A.c2, c3, A.key0, A.key1);
            pairs4(a.w[j], b.w[j], ea.w[j], eb.w[j], rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, s_thr, a3);
          }
          sigma_sums(a, aF, aT); sigma_sums(b, bF, bT);
          st16(gpb + 8 * v * SEG + X0, b);                                       // plane row (ky, kb): 8 rows below for v = 1
          if (sh_a == 0) st16(gpa + 8 * v * SEG + X0, a);
          else st16_left1_tile(gpa + 8 * v * SEG, reinterpret_cast<uint8_t*>(mp->pl) + 8 * v * SEG, X0, a);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s));
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
