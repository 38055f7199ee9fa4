// ic_kernels_staged.cuh -- variant 3: the production sm_100a kernels for L >= 2048 on the tiled layout LAY_P16.
//
// One launch = one phase of a sweep (schedule S1, U4), one persistent block per SM, launched as a programmatic
// dependent of the previous kernel of the stream (table fill and barrier set-up overlap that kernel's tail):
//   * 4 producer warps stage "regions" of the lattice in shared memory with 1-D bulk copies (cp.async.bulk, the TMA
//     engine; completion on an mbarrier).  A region is one tile of the layout (row quad Y, 512 plane columns: 16 plane
//     rows = 8 KB contiguous in global memory, ONE copy) plus the plane rows of the lattice row above and of the one
//     (NEAR-V: two) below (2 KB / 4 KB contiguous, one copy each).  The few bytes read across the left/right tile
//     edge (the x-1 neighbour of plane 0 is plane 3 one byte to the left) are fetched by the producer's other lanes
//     with plain loads into a small side array.  Bulk copies cost ~120 cycles of issue each whatever their size
//     (measured), which is why the layout makes a region three copies and not twenty.
//   * 24 consumer warps in 3 groups; group g processes tasks g, g+3, ... of the block and owns two stage slots
//     (double buffering; a slot goes back to the producer as soon as the items are in registers).  A task is two
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

constexpr int ST_GROUPS = 3;                  // consumer groups per block
constexpr int ST_NPROD = 4;                   // producer warps per block
constexpr int ST_LOGSEG = P16_LOGSEG_MAX, ST_SEG = 1 << ST_LOGSEG;   // plane columns per region = per tile of the layout
constexpr int ST_TPG = ST_SEG / 2;            // consumer threads per group: one 16-pair item each per task
constexpr int ST_THREADS = 32 * ST_NPROD + ST_GROUPS * ST_TPG;
constexpr int ST_DESC_ENTRIES = 256;          // move descriptors [key*8 + r] (224 used) in global memory: (coefficients, info)
constexpr int ST_DESC_SMEM = 28 * 8 * 128;    // in shared memory: [key][r][lane & 15] x 8 bytes, a private copy per lane

template <int TYPE>
struct StagedCfg {
  static constexpr int ROWS = TYPE == PH_NEAR_V ? 28 : 24;          // staged plane rows: (ky_rel + 1) * 4 + kx, ky_rel = -1..4 (5)
  static constexpr int REGION_BYTES = ROWS * ST_SEG;
  static constexpr int OFF_HALO = 2 * REGION_BYTES;                 // uint8 [2 regions][left, right][32 rows]
  static constexpr int OFF_SMETA = OFF_HALO + 128;                  // SubMeta[4]
  static constexpr int STAGE_BYTES = OFF_SMETA + 256;
  static constexpr int NSTAGE = 2 * ST_GROUPS;                       // two ring slots per consumer group (see the kernel)
  static constexpr int TASK_TX = 2 * (16 + 4 + (ROWS - 20)) * ST_SEG;   // bytes the bulk copies of one task deliver
  // dynamic shared memory map (byte offsets)
  static constexpr int OFF_THR = 0;                                 // uint32 threshold[THR_STRIDE], then uint32 packed deltas[THR_STRIDE]
  static constexpr int OFF_DESC = OFF_THR + THR_STRIDE * 8;         // uint2 descriptors [28][8][16]
  static constexpr int OFF_STAGE = OFF_DESC + ST_DESC_SMEM;         // NSTAGE stage buffers
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
// producers are far ahead of the consumers most of the time: sleep between polls instead of burning issue slots
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    if (ok) break;
    __nanosleep(400);
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
//   move descriptor [key][r], key = fa | fb<<1 | ga<<3 | gb<<4, r = w & 7 (the table of two-site configurations,
//   PAPER.md:66-74), 8 bytes, 16 copies so that every lane of a half warp reads its own banks (no conflicts at all):
//   coef = four int8 coefficients;  info = shared-memory address of the class base in the threshold table (low 16 bits) |
//   xor of the site bytes (a at bits 0,3; b at bits 1,4) << 16.
//   class tables [class]: threshold 8*t29 - 1 (accept iff w <= it), packed (dn2, dV, dJ).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lds_tab32(uint32_t addr) {
  uint32_t v;
  asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void pairs4(uint32_t& A4, uint32_t& B4, uint32_t EA4, uint32_t EB4, uint32_t w0, uint32_t w1,
                                       uint32_t w2, uint32_t w3, uint32_t s_desc, int& a3) {
  // neighbour sums as (4F, 8G), G coefficients halved: the dp4a below yields a byte address in the 4-byte thresholds
  const uint32_t FA = (EA4 << 2) & 0x1C1C1C1Cu, GA = EA4 & 0x38383838u;
  const uint32_t FB = (EB4 << 2) & 0x1C1C1C1Cu, GB = EB4 & 0x38383838u;
  const uint32_t t0 = __byte_perm(FA, GA, 0x5140), t1 = __byte_perm(FA, GA, 0x7362);
  const uint32_t u0 = __byte_perm(FB, GB, 0x5140), u1 = __byte_perm(FB, GB, 0x7362);
  const uint32_t W0 = __byte_perm(t0, u0, 0x5410), W1 = __byte_perm(t0, u0, 0x7632);
  const uint32_t W2 = __byte_perm(t1, u1, 0x5410), W3 = __byte_perm(t1, u1, 0x7632);
  // key fa | fb<<1 | ga<<3 | gb<<4 (< 28), times 4 in each byte; byte i moved to byte 1 is key * 1024 = its table row
  const uint32_t KS = 4u * A4 + 8u * B4;
  const uint2 q0 = lds_tab64(s_desc + __byte_perm(KS, 0u, 0x4404) + ((w0 & 7u) << 7));   // s_desc includes (lane & 15) * 8
  const uint2 q1 = lds_tab64(s_desc + __byte_perm(KS, 0u, 0x4414) + ((w1 & 7u) << 7));
  const uint2 q2 = lds_tab64(s_desc + __byte_perm(KS, 0u, 0x4424) + ((w2 & 7u) << 7));
  const uint2 q3 = lds_tab64(s_desc + __byte_perm(KS, 0u, 0x4434) + ((w3 & 7u) << 7));
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
// grid = (blocks, replicas), block = 4 producer warps + 4 groups of 128 consumer threads.
// ---------------------------------------------------------------------------------------------------------------
template <int TYPE, int CW>
__global__ void __launch_bounds__(ST_THREADS, 1) k_staged_phase(PhaseArgs A) {
  using C = StagedCfg<TYPE>;
  constexpr int SEG = ST_SEG, LOGSEG = ST_LOGSEG, NST = C::NSTAGE;
  extern __shared__ __align__(128) unsigned char smem[];
  const int r = blockIdx.y, tid = threadIdx.x, lane = tid & 31;
  const uint32_t bar0 = smem_u32(smem + C::OFF_BAR);                    // full[s] at bar0 + 8 s, empty[s] at + 8 (NST + s)
  // Programmatic dependent launch: the next kernel of the stream may start its blocks as soon as ours leave their SMs;
  // it fills its tables (which no kernel writes) and then waits for the whole of this grid before touching the lattice.
  asm volatile("griddepcontrol.launch_dependents;");
  {
    const uint2* src = A.thr + (long long)r * THR_STRIDE;
    uint32_t* thr_s = reinterpret_cast<uint32_t*>(smem + C::OFF_THR);
    for (int k = tid; k < THR_STRIDE; k += ST_THREADS) { const uint2 v = __ldg(&src[k]); thr_s[k] = v.x; thr_s[THR_STRIDE + k] = v.y; }
    const uint2* dsrc = A.desc32 + (TYPE == PH_FAR ? 0 : ST_DESC_ENTRIES);
    uint2* desc_s = reinterpret_cast<uint2*>(smem + C::OFF_DESC);
    for (int k = tid; k < ST_DESC_SMEM / 8; k += ST_THREADS) {
      const int key = k >> 7, rr = (k >> 4) & 7;               // keys with bit 2 set do not occur: null entries
      uint2 d = __ldg(&dsrc[key * 8 + rr]);
      d.y += smem_u32(smem + C::OFF_THR);       // low 16 bits: shared-memory address of the class base (< 64 KB)
      desc_s[k] = d;
    }
    if (tid == 0) {
      for (int s = 0; s < NST; ++s) {
        mbar_init(bar0 + 8 * s, 2);                                     // producer lane 0: expect_tx, and after the edge bytes
        mbar_init(bar0 + 8 * (NST + s), ST_TPG / 32);                   // the warps of the consuming group
      }
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");                    // the previous phase / fold kernel is complete
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
  // tasks of this block: t = blockIdx.x + n * gridDim.x, n = 0, 1, ...; task n belongs to consumer group g = n % ST_GROUPS
  // and is its k-th task, k = n / ST_GROUPS; it lives in slot g + ST_GROUPS * (k & 1) on lap (k >> 1) & 1.  A slot is thus
  // always drained by the same group and filled by the same producer warp, both in task order, so nobody can wait on a
  // barrier more than one phase away from its own -- the only case a parity wait gets wrong.  (With slots shared between
  // groups a group that ran a lap ahead of a slow producer passed the wait on the previous lap's parity.)
  int tn2 = 0, tV = 0, tJ = 0, tM = 0, tMs = 0;
  int aF = 0, aT = 0, bF = 0, bT = 0, sgn = 1;   // sums over the new site bytes of the a- and b-sites (sigma_sums)

  if (tid < 32 * ST_NPROD) {
    // ============================== producer warps: warp p fills the ring slots s with s % ST_NPROD == p ================
    const int p = tid >> 5;
    const int hf = lane < C::ROWS ? halo_flags(TYPE, A.phase, A.p2, (lane >> 2) - 1, lane & 3) : 0;   // lane = staged row
    // a slot is always filled by the same producer warp (slot % ST_NPROD), in task order
    for (int t = blockIdx.x, g = 0, k = 0; t < ntasks; t += gridDim.x, k += (g + 1 == ST_GROUPS), g = (g + 1 == ST_GROUPS) ? 0 : g + 1) {
      const int s = g + ST_GROUPS * (k & 1), lap = (k >> 1) & 1;
      if (s % ST_NPROD != p) continue;
      mbar_wait_backoff(bar0 + 8 * (NST + s), (uint32_t)(lap ^ 1));
      unsigned char* stg = smem + C::OFF_STAGE + s * C::STAGE_BYTES;
      const uint32_t full = bar0 + 8 * s;
      int Yq[2], sg[2];
#pragma unroll
      for (int U = 0; U < 2; ++U) { const int rho = region_of(t, U); Yq[U] = rho >> lognseg; sg[U] = rho & (nseg - 1); }
      // bytes across the tile edge (lane = staged row (ky_rel + 1) * 4 + kx): plain loads, issued first so that their
      // latency overlaps with the issue of the bulk copies
      uint8_t hl[2] = {0, 0}, hr[2] = {0, 0};
      if (hf) {
        const int kyr = (lane >> 2) - 1, kx = lane & 3, ky = kyr & 3;
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          const int Yr = kyr < 0 ? ((Yq[U] - 1) & Wm) : kyr > 3 ? ((Yq[U] + 1) & Wm) : Yq[U];
          if (hf & 1) hl[U] = lat[p16_row(lw, ky, kx, Yr, (sg[U] - 1) & (nseg - 1)) + SEG - 1];
          if (hf & 2) hr[U] = lat[p16_row(lw, ky, kx, Yr, (sg[U] + 1) & (nseg - 1))];
        }
      }
      if (lane == 0) {
        mbar_arrive_expect_tx(full, (uint32_t)C::TASK_TX);
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          const uint32_t dst = smem_u32(stg + U * C::REGION_BYTES);
          bulk_g2s(dst + 4 * SEG, lat + p16_row(lw, 0, 0, Yq[U], sg[U]), 16 * SEG, full);
          bulk_g2s(dst, lat + p16_row(lw, 3, 0, (Yq[U] - 1) & Wm, sg[U]), 4 * SEG, full);
          bulk_g2s(dst + 20 * SEG, lat + p16_row(lw, 0, 0, (Yq[U] + 1) & Wm, sg[U]), (C::ROWS - 20) * SEG, full);
        }
      }
      if (lane >= 28) {
        // sub-task (U, half): where its items store to, and the coordinates for the Philox counters
        const int sub = lane - 28, U = sub >> 1, half = sub & 1, Y = Yq[U], seg = sg[U];
        SubMeta mt; mt.Y = Y; mt.S0 = seg << LOGSEG; mt.pl = 0ull;
        if (TYPE == PH_FAR) {
          const int UP = paired ? (U ^ 1) : U;
          const int ky = A.phase + 2 * half, kyb = ky ^ (my & 3);
          mt.pa = (unsigned long long)(lat + p16_row(lw, ky, 0, Y, seg));
          mt.pb = (unsigned long long)(lat + p16_row(lw, kyb, 0, Yq[UP], sg[UP]));
        } else if (TYPE == PH_NEAR_V) {
          const int ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kyb = (ky + 1) & 3, Yb = (Y + (ky == 3)) & Wm;
          mt.pa = (unsigned long long)(lat + p16_row(lw, ky, 0, Y, seg));
          mt.pb = (unsigned long long)(lat + p16_row(lw, kyb, 0, Yb, seg));
        } else {
          const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
          mt.pa = (unsigned long long)(lat + p16_row(lw, half, ka, Y, seg));
          mt.pb = (unsigned long long)(lat + p16_row(lw, half, kb, Y, seg));
          mt.pl = (unsigned long long)(lat + p16_row(lw, half, ka, Y, (seg - 1) & (nseg - 1)) + SEG - 1);
        }
        SubMeta* dstm = reinterpret_cast<SubMeta*>(stg + C::OFF_SMETA) + sub;
        dstm->pa = mt.pa; dstm->pb = mt.pb; dstm->pl = mt.pl; dstm->Y = mt.Y; dstm->S0 = mt.S0;
      }
      if (hf) {
#pragma unroll
        for (int U = 0; U < 2; ++U) {
          if (hf & 1) stg[C::OFF_HALO + U * 64 + lane] = hl[U];
          if (hf & 2) stg[C::OFF_HALO + U * 64 + 32 + lane] = hr[U];
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(full);
    }
  } else {
    // =========================================== consumer warps ====================================================
    const int ct = tid - 32 * ST_NPROD, g = ct / ST_TPG, tg = ct - g * ST_TPG;
    // item = one 16-byte vector of a-sites (b-sites for NEAR-H) = 16 coupled pairs: sub-task (U, half), plane/row selector
    // hi, chunk of 16 plane columns (SEG / 16 = 32 chunks); all but the chunk are uniform in a warp
    const int sub = tg >> 6, hi = (tg >> 5) & 1, chunk = tg & 31, U = sub >> 1, half = sub & 1, X0 = chunk << 4;
    const uint32_t s_desc = smem_u32(smem + C::OFF_DESC) + (uint32_t)(lane & 15) * 8u;
    const uint32_t c3 = (uint32_t)r | (TAG_UPDATE << 28);
    auto addf = [](const V16& p, const V16& q) -> V16 { return add(p, q); };
    // byte offsets inside a stage buffer: the 16 bytes at plane column Xc of staged row (ky_rel, kx) of region UU,
    // and the bytes just left / right of them (across the tile edge: the side array filled by the producer)
    auto off = [&](int UU, int kyr, int kx, int Xc) -> int { return UU * C::REGION_BYTES + ((((kyr + 1) << 2) + (kx & 3)) << LOGSEG) + Xc; };
    auto offL = [&](int UU, int kyr, int kx, int Xc) -> int {
      return Xc ? off(UU, kyr, kx, Xc) - 1 : C::OFF_HALO + UU * 64 + ((kyr + 1) << 2) + (kx & 3);
    };
    auto offR = [&](int UU, int kyr, int kx, int Xc) -> int {
      return Xc != SEG - 16 ? off(UU, kyr, kx, Xc) + 16 : C::OFF_HALO + UU * 64 + 32 + ((kyr + 1) << 2) + (kx & 3);
    };
    // FAR: byte part of the lane permutation i -> i ^ (mx >> 2 & 15) as a PRMT selector (index b -> b ^ (c & 3))
    const uint32_t selb = 0x3210u ^ (0x1111u * (uint32_t)((mx >> 2) & 3));
    for (int t = blockIdx.x + g * gridDim.x, k = 0; t < ntasks; t += ST_GROUPS * gridDim.x, ++k) {
      const int s = g + ST_GROUPS * (k & 1), lap = (k >> 1) & 1;
      mbar_wait(bar0 + 8 * s, (uint32_t)lap);
      const uint8_t* st = smem + C::OFF_STAGE + s * C::STAGE_BYTES;
      const SubMeta* mp = reinterpret_cast<const SubMeta*>(st + C::OFF_SMETA) + sub;
      const int Y = mp->Y, chunkG = (mp->S0 >> 4) + chunk;
      uint8_t* gpa = reinterpret_cast<uint8_t*>(mp->pa);
      uint8_t* gpb = reinterpret_cast<uint8_t*>(mp->pb);
      // the 16 bytes of plane kx at row kyr, shifted by one site to the left (sh < 0) or right (sh > 0) if asked
      auto ldrow = [&](int UU, int kyr, int kx, int Xc, int sh) -> V16 {
        V16 v = ld16(st + off(UU, kyr, kx, Xc));
        if (sh < 0) v = shift_up(v, st[offL(UU, kyr, kx, Xc)]);
        else if (sh > 0) v = shift_down(v, st[offR(UU, kyr, kx, Xc)]);
        return v;
      };
      // left + right neighbours of the vector of plane kx: planes kx-1 and kx+1, one site over when they wrap around
      auto xsum = [&](int UU, int kyr, int kx, int Xc) -> V16 {
        return addf(ldrow(UU, kyr, kx + 3, Xc, kx == 0 ? -1 : 0), ldrow(UU, kyr, kx + 1, Xc, kx == 3 ? 1 : 0));
      };
      V16 a, b, ea, eb;
      int y, kxr;                       // Philox counters: lattice row and plane of the slot site
      bool left1 = false;               // NEAR-H with ka = 3: the a-vector starts one plane column to the left
      uint8_t* gpl = nullptr;
      if (TYPE == PH_FAR) {
        const int ky = A.phase + 2 * half, kxa = 2 * hi;
        const int kyb = ky ^ (my & 3), UB = paired ? (U ^ 1) : U, kxb = kxa ^ (mx & 3);
        const int Xb = X0 ^ ((mx >> 2) & (SEG - 1) & ~15);               // the partner chunk inside the partner tile
        sgn = A.phase ? -1 : 1;
        a = ld16(st + off(U, ky, kxa, X0));
        ea = addf(xsum(U, ky, kxa, X0), addf(ld16(st + off(U, ky - 1, kxa, X0)), ld16(st + off(U, ky + 1, kxa, X0))));
        b = ld16(st + off(UB, kyb, kxb, Xb));
        eb = addf(xsum(UB, kyb, kxb, Xb), addf(ld16(st + off(UB, kyb - 1, kxb, Xb)), ld16(st + off(UB, kyb + 1, kxb, Xb))));
        b = xor_perm<CW>(b, selb); eb = xor_perm<CW>(eb, selb);          // b into a's lane order (lane i <-> i ^ c)
        y = 4 * Y + ky; kxr = kxa;
        gpa += kxa * SEG + X0; gpb += kxb * SEG + Xb;
      } else if (TYPE == PH_NEAR_V) {
        const int kx = half + 2 * hi, ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3;
        sgn = ((half + ky) & 1) ? -1 : 1;
        a = ld16(st + off(U, ky, kx, X0)); b = ld16(st + off(U, ky + 1, kx, X0));     // row 4 = row 0 of the quad below
        // vertical domino: a's lower neighbour is b, b's upper neighbour is a
        ea = addf(xsum(U, ky, kx, X0), addf(ld16(st + off(U, ky - 1, kx, X0)), b));
        eb = addf(xsum(U, ky + 1, kx, X0), addf(a, ld16(st + off(U, ky + 2, kx, X0))));
        y = 4 * Y + ky; kxr = kx;
        gpa += kx * SEG + X0; gpb += kx * SEG + X0;
      } else {
        // NEAR, horizontal dominoes of row ky = half + 2 hi; lanes are indexed by the b-site
        const int ky = half + 2 * hi;
        const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
        const int sh_a = -(ka == 3), sh_l = sh_a - (ka == 0), sh_r = (kb == 3);
        sgn = ((ka + half) & 1) ? -1 : 1;
        a = ldrow(U, ky, ka, X0, sh_a); b = ld16(st + off(U, ky, kb, X0));
        ea = addf(addf(ldrow(U, ky, ka + 3, X0, sh_l), b), addf(ldrow(U, ky - 1, ka, X0, sh_a), ldrow(U, ky + 1, ka, X0, sh_a)));
        eb = addf(addf(a, ldrow(U, ky, kb + 1, X0, sh_r)), addf(ld16(st + off(U, ky - 1, kb, X0)), ld16(st + off(U, ky + 1, kb, X0))));
        y = 4 * Y + ky; kxr = kb;
        left1 = sh_a != 0;
        gpa += 8 * hi * SEG; gpb += 8 * hi * SEG + X0;                           // plane rows (ky, ka), (ky, kb)
        gpl = reinterpret_cast<uint8_t*>(mp->pl) + 8 * hi * SEG;
      }
      // everything the item needs is in registers: hand the ring slot back to the producer before the long part
      __syncwarp();
      if (lane == 0) mbar_arrive(bar0 + 8 * (NST + s));
      // random words: block c0 = 4*(X>>2) + kx, c1 = y, word X & 3 of the slot site (U3)
      int a3 = 0;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const u32x4 rr = philox4x32_10((uint32_t)(4 * (4 * chunkG + j) + kxr), (uint32_t)y, A.c2, c3, A.key0, A.key1);
        pairs4(a.w[j], b.w[j], ea.w[j], eb.w[j], rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, a3);
      }
      if (TYPE == PH_FAR) b = xor_perm<CW>(b, selb);
      sigma_sums(a, aF, aT); sigma_sums(b, bF, bT);
      st16(gpb, b);
      if (TYPE == PH_NEAR_H) { if (!left1) st16(gpa + X0, a); else st16_left1_tile(gpa, gpl, X0, a); }
      else st16(gpa, a);
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
