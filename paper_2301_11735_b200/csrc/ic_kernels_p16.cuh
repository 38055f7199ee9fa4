// ic_kernels_p16.cuh -- variant 2: the tiled sm_100a kernels on the tiled layout LAY_P16 for 64 <= L <= 2048 (one tile
// per row quad: a plane row is a whole lattice row), vectors loaded straight from global memory.  Also the home of the
// 16-byte vector helpers (with the widen / pack of the 2-bit layout LAY_P2) and the layout converters that the staged and
// one-launch kernels (ic_kernels_staged.cuh, ic_kernels_coop.cuh) share.
//
// One phase of a sweep = one launch.  In every phase of schedule S1 the a-sites and the b-sites are whole plane rows
// [y&3][x&3] of the layout, so a thread works on dense 16-byte vectors: an "item" is two vectors of 16 coupled pairs
// (32 pair updates), eight Philox4x32-7 blocks.  Per item:
//   1. 128-bit loads of the a- and b-vectors and of their neighbour vectors (A2 of SURVEY 8(a)); the neighbour sums
//      of 4 sites are byte-wise 32-bit adds: byte = F | G<<3, sum S = F+G-4, sum sigma = F-G;
//   2. per 4 pairs: a 4x4 byte transpose gives W_i = (8Fa, 8Ga, 8Fb, 8Gb); the pair key (fa,fb,ga,gb) and the
//      3 proposal bits of the pair's random word index a 64-bit move descriptor in shared memory (the table of
//      two-site configurations of PAPER.md:66-74 -- the paper keeps it in constant memory);
//   3. one dp4a gives the byte offset of the dE class (eq. 4/5, linear in the neighbour sums),
//      one 64-bit shared load gives (threshold, packed (dn2,dV,dJ)); accept iff w <= threshold;
//   4. accepted moves xor their change into the vectors; vectors are stored back with 128-bit stores;
//   5. observables: per-thread packed integer sums -> warp REDUX -> block -> one int64 atomic per value (A8).
#pragma once
#include "ic_common.cuh"
#include "ic_kernels_ref.cuh"

namespace ic {

constexpr int DESC_ENTRIES = 28 * 8;          // key (fa | fb<<1 | ga<<3 | gb<<4) in 0..27, proposal r in 0..7
constexpr int P16_THREADS = 256;

enum { PH_FAR = 0, PH_NEAR_H = 1, PH_NEAR_V = 2 };

struct V16 { uint32_t w[4]; };

__device__ __forceinline__ V16 ld16(const uint8_t* p) {
  const uint4 v = *reinterpret_cast<const uint4*>(p);
  V16 r; r.w[0] = v.x; r.w[1] = v.y; r.w[2] = v.z; r.w[3] = v.w; return r;
}
__device__ __forceinline__ void st16(uint8_t* p, const V16& v) {
  *reinterpret_cast<uint4*>(p) = make_uint4(v.w[0], v.w[1], v.w[2], v.w[3]);
}
// LAY_P2 (ic_common.cuh): a 32-bit word of 16 sites <-> the 16-byte vector of site bytes f | g<<3
__device__ __forceinline__ V16 widen2(uint32_t w) {
  V16 r;
  r.w[0] = w & 0x09090909u; r.w[1] = __funnelshift_r(w, w, 2) & 0x09090909u;
  r.w[2] = __funnelshift_r(w, w, 4) & 0x09090909u; r.w[3] = __funnelshift_r(w, w, 6) & 0x09090909u;
  return r;
}
__device__ __forceinline__ uint32_t pack2(const V16& v) {          // bytes must be clean (bits 0 and 3 only)
  return v.w[0] | __funnelshift_l(v.w[1], v.w[1], 2) | __funnelshift_l(v.w[2], v.w[2], 4) | __funnelshift_l(v.w[3], v.w[3], 6);
}
// the vector / the site byte at the P16 byte offset `off` of a lattice in either tiled layout (off = site index in P2)
template <int BITS>
__device__ __forceinline__ V16 ldvec(const uint8_t* lat, long long off) {
  if (BITS == 8) return ld16(lat + off);
  return widen2(*reinterpret_cast<const uint32_t*>(lat + (off >> 2)));
}
template <int BITS>
__device__ __forceinline__ uint32_t ldsite(const uint8_t* lat, long long off) {
  if (BITS == 8) return lat[off];
  return (uint32_t)p2_site_e(*reinterpret_cast<const uint32_t*>(lat + ((off >> 4) << 2)), (int)(off & 15));
}
__device__ __forceinline__ V16 add(const V16& a, const V16& b) {   // byte-wise: every byte <= 36, no carries
  V16 r;
#pragma unroll
  for (int k = 0; k < 4; ++k) r.w[k] = a.w[k] + b.w[k];
  return r;
}
// bytes (e, v0 .. v14): the vector one site to the left
__device__ __forceinline__ V16 shift_up(const V16& v, uint32_t e) {
  V16 r;
  r.w[3] = __funnelshift_l(v.w[2], v.w[3], 8); r.w[2] = __funnelshift_l(v.w[1], v.w[2], 8);
  r.w[1] = __funnelshift_l(v.w[0], v.w[1], 8); r.w[0] = (v.w[0] << 8) | e;
  return r;
}
// bytes (v1 .. v15, e): the vector one site to the right
__device__ __forceinline__ V16 shift_down(const V16& v, uint32_t e) {
  V16 r;
  r.w[0] = __funnelshift_r(v.w[0], v.w[1], 8); r.w[1] = __funnelshift_r(v.w[1], v.w[2], 8);
  r.w[2] = __funnelshift_r(v.w[2], v.w[3], 8); r.w[3] = (v.w[3] >> 8) | (e << 24);
  return r;
}
// 16 bytes of a plane row starting at X0 + sh (sh in {-1,0,+1}), periodic in the row of W bytes
__device__ __forceinline__ V16 ldrow(const uint8_t* row, int X0, int W, int sh) {
  V16 v = ld16(row + X0);
  if (sh < 0) v = shift_up(v, row[(X0 - 1) & (W - 1)]);
  else if (sh > 0) v = shift_down(v, row[(X0 + 16) & (W - 1)]);
  return v;
}
// store 16 bytes at X0 - 1 .. X0 + 14 (periodic): byte-granular so that neighbouring threads never share a store
__device__ __forceinline__ void st16_left1(uint8_t* row, int X0, int W, const V16& v) {
  row[(X0 - 1) & (W - 1)] = (uint8_t)(v.w[0] & 0xFFu);
  const V16 s = shift_down(v, 0u);                       // bytes v1..v15 at X0..X0+14
  *reinterpret_cast<uint2*>(row + X0) = make_uint2(s.w[0], s.w[1]);
  *reinterpret_cast<uint32_t*>(row + X0 + 8) = s.w[2];
  *reinterpret_cast<uint16_t*>(row + X0 + 12) = (uint16_t)(s.w[3] & 0xFFFFu);
  row[X0 + 14] = (uint8_t)((s.w[3] >> 16) & 0xFFu);
}
// lane permutation i -> i ^ c inside a 16-byte vector; CW = c >> 2 (compile time), selb = byte selector for c & 3
template <int CW>
__device__ __forceinline__ V16 xor_perm(const V16& v, uint32_t selb) {
  V16 r;
#pragma unroll
  for (int k = 0; k < 4; ++k) r.w[k] = __byte_perm(v.w[k ^ CW], 0u, selb);
  return r;
}

struct ItemAcc { int a3; int m16; int d16; };

// Four coupled pairs: site bytes A4/B4, neighbour-sum bytes EA4/EB4, one random word per pair.
__device__ __forceinline__ void process4(uint32_t& A4, uint32_t& B4, uint32_t EA4, uint32_t EB4,
                                         uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3,
                                         const char* s_desc, const char* s_thr, ItemAcc& acc) {
  // lanes scaled by 8: the dp4a below yields a byte offset into the table of 8-byte class entries
  const uint32_t FA = (EA4 << 3) & 0x38383838u, GA = EA4 & 0x38383838u;
  const uint32_t FB = (EB4 << 3) & 0x38383838u, GB = EB4 & 0x38383838u;
  const uint32_t t0 = __byte_perm(FA, GA, 0x5140), t1 = __byte_perm(FA, GA, 0x7362);
  const uint32_t u0 = __byte_perm(FB, GB, 0x5140), u1 = __byte_perm(FB, GB, 0x7362);
  const uint32_t W0 = __byte_perm(t0, u0, 0x5410), W1 = __byte_perm(t0, u0, 0x7632);
  const uint32_t W2 = __byte_perm(t1, u1, 0x5410), W3 = __byte_perm(t1, u1, 0x7632);
  const uint32_t KEY = A4 + 2u * B4;                      // per byte: fa | fb<<1 | ga<<3 | gb<<4
  uint32_t D4 = 0u, MD4 = 0u;
#define IC_PAIR(i, Wi, wi, SELD, SELM)                                                                              \
  {                                                                                                                 \
    const uint32_t koff = ((i) == 0 ? (KEY << 6) : (KEY >> (8 * (i) - 6))) & 0x6C0u;                                \
    const uint2 d = *reinterpret_cast<const uint2*>(s_desc + (koff | (((wi) & 7u) << 3)));                          \
    const int off = __dp4a((int)(Wi), (int)d.x, (int)(d.y & 0x7FFFu));                                              \
    const uint2 c = *reinterpret_cast<const uint2*>(s_thr + off);                                                   \
    if ((wi) <= c.x) {                                                                                              \
      acc.a3 += (int)c.y;                                                                                           \
      D4 = __byte_perm(D4, d.y, SELD);                                                                              \
      MD4 = __byte_perm(MD4, d.y, SELM);                                                                            \
    }                                                                                                               \
  }
  IC_PAIR(0, W0, w0, 0x3216, 0x3217)
  IC_PAIR(1, W1, w1, 0x3260, 0x3270)
  IC_PAIR(2, W2, w2, 0x3610, 0x3710)
  IC_PAIR(3, W3, w3, 0x6210, 0x7210)
#undef IC_PAIR
  A4 ^= D4 & 0x09090909u;
  B4 ^= (D4 >> 1) & 0x09090909u;
  acc.m16 = __dp4a((int)((MD4 << 4) & 0xF0F0F0F0u), 0x01010101, acc.m16);   // 16 * sum (dsig_a + dsig_b)
  acc.d16 = __dp4a((int)(MD4 & 0xF0F0F0F0u), 0x01010101, acc.d16);          // 16 * sum (dsig_a - dsig_b)
}

// left+right neighbour sums of the two vectors (kx = sel, sel+2) of one lattice row, from the two other planes of the row
__device__ __forceinline__ void xnbr_sums(const uint8_t* lat, int lw, int W, int ky, int Y, int sel, int X0, V16& s_lo, V16& s_hi) {
  const uint8_t* r0 = lat + p16_row(lw, ky, sel + 1, Y, 0);             // plane between lo and hi
  const uint8_t* r1 = lat + p16_row(lw, ky, (sel + 3) & 3, Y, 0);     // plane right of hi / left of lo
  const V16 q0 = ld16(r0 + X0), q1 = ld16(r1 + X0);
  if (sel == 0) { s_lo = add(q0, shift_up(q1, r1[(X0 - 1) & (W - 1)])); s_hi = add(q0, q1); }
  else { s_lo = add(q0, q1); s_hi = add(q0, shift_down(q1, r1[(X0 + 16) & (W - 1)])); }
}

__device__ __forceinline__ const uint8_t* rowptr(const uint8_t* lat, int lw, int ky, int kx, int Y) {
  return lat + p16_row(lw, ky, kx, Y, 0);     // lw <= 9: one tile per row quad, a plane row is a whole lattice row
}

template <int TYPE, int CW>
__global__ void __launch_bounds__(P16_THREADS) k_p16_phase(PhaseArgs A) {
  __shared__ __align__(16) uint2 s_thr_tab[THR_STRIDE];
  __shared__ __align__(16) uint2 s_desc_tab[DESC_ENTRIES];
  const int r = blockIdx.y;
  asm volatile("griddepcontrol.launch_dependents;");      // programmatic dependent launch: see launch_pdl (ic_api.cu)
  {
    const uint4* src = reinterpret_cast<const uint4*>(A.thr + (long long)r * THR_STRIDE);
    uint4* dst = reinterpret_cast<uint4*>(s_thr_tab);
    for (int k = threadIdx.x; k < THR_STRIDE / 2; k += P16_THREADS) dst[k] = __ldg(&src[k]);
    if (threadIdx.x < DESC_ENTRIES) s_desc_tab[threadIdx.x] = __ldg(&A.desc[threadIdx.x]);
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");      // the tables above are written by no kernel
  __syncthreads();
  const char* s_thr = reinterpret_cast<const char*>(s_thr_tab);
  const char* s_desc = reinterpret_cast<const char*>(s_desc_tab);

  const int lw = A.logL - 2, W = 1 << lw, Wm = W - 1;
  const int lognch = lw - 4, nch = 1 << lognch;
  const long long n_items = (long long)W * 2 * nch;
  uint8_t* lat = reinterpret_cast<uint8_t*>(A.lattice) + (long long)r * A.lat_stride;
  const uint32_t c3 = (uint32_t)r | (TAG_UPDATE << 28);
  int tn2 = 0, tV = 0, tJ = 0, tM = 0, tMs = 0;

  for (long long id = (long long)blockIdx.x * P16_THREADS + threadIdx.x; id < n_items; id += (long long)gridDim.x * P16_THREADS) {
    const int chunk = (int)(id & (nch - 1)), half = (int)(id >> lognch) & 1, Y = (int)(id >> (lognch + 1));
    const int X0 = chunk << 4;
    ItemAcc acc; acc.a3 = 0; acc.m16 = 0; acc.d16 = 0;
    int sgn;

    if (TYPE == PH_FAR || TYPE == PH_NEAR_V) {
      // ---- two a-vectors (kx = sel, sel+2) of lattice row y = 4Y + ky, partners in row (kyb, Yb) --------------------
      int sel, ky, kyb, Yb, Xb0, selb_planes;
      uint32_t selb = 0x3210u;
      if (TYPE == PH_FAR) {
        const int mx = A.p1, my = A.p2;
        sel = 0; ky = A.phase + 2 * half;
        kyb = ky ^ (my & 3); Yb = Y ^ (my >> 2); Xb0 = X0 ^ ((mx >> 2) & ~15);
        selb_planes = 1;                                   // b-vectors are the planes kx = 1, 3 of row (kyb, Yb)
        const int cb = (mx >> 2) & 3;
        selb = cb == 0 ? 0x3210u : cb == 1 ? 0x2301u : cb == 2 ? 0x1032u : 0x0123u;
        sgn = A.phase ? -1 : 1;
      } else {
        sel = half; ky = (A.p2 + 2 * ((half + A.phase) & 1)) & 3;
        kyb = (ky + 1) & 3; Yb = (Y + (ky == 3)) & Wm; Xb0 = X0;
        selb_planes = sel;
        sgn = ((sel + ky) & 1) ? -1 : 1;
      }
      const int y = 4 * Y + ky;
      // a side
      uint8_t* pa_lo = const_cast<uint8_t*>(rowptr(lat, lw, ky, sel, Y)) + X0;
      uint8_t* pa_hi = const_cast<uint8_t*>(rowptr(lat, lw, ky, sel + 2, Y)) + X0;
      V16 a_lo = ld16(pa_lo), a_hi = ld16(pa_hi);
      V16 ea_lo, ea_hi;
      xnbr_sums(lat, lw, W, ky, Y, sel, X0, ea_lo, ea_hi);
      {
        const int kyu = (ky - 1) & 3, Yu = (Y - (ky == 0)) & Wm;
        ea_lo = add(ea_lo, ld16(rowptr(lat, lw, kyu, sel, Yu) + X0));
        ea_hi = add(ea_hi, ld16(rowptr(lat, lw, kyu, sel + 2, Yu) + X0));
      }
      // b side, natural lane order
      int kxb_lo, kxb_hi;
      if (TYPE == PH_FAR) { kxb_lo = (A.p1 & 3); kxb_hi = 2 ^ (A.p1 & 3); }     // partner planes of kx = 0 and kx = 2
      else { kxb_lo = sel; kxb_hi = sel + 2; }
      uint8_t* pb_lo = const_cast<uint8_t*>(rowptr(lat, lw, kyb, kxb_lo, Yb)) + Xb0;
      uint8_t* pb_hi = const_cast<uint8_t*>(rowptr(lat, lw, kyb, kxb_hi, Yb)) + Xb0;
      V16 b_lo = ld16(pb_lo), b_hi = ld16(pb_hi);
      V16 eb_lo, eb_hi;
      {
        V16 s_first, s_second;                              // sums for planes (selb_planes, selb_planes + 2)
        xnbr_sums(lat, lw, W, kyb, Yb, selb_planes, Xb0, s_first, s_second);
        if (TYPE == PH_FAR) { const bool sw = (kxb_lo == 3); eb_lo = sw ? s_second : s_first; eb_hi = sw ? s_first : s_second; }
        else { eb_lo = s_first; eb_hi = s_second; }
        const int kyd = (kyb + 1) & 3, Yd = (Yb + (kyb == 3)) & Wm;
        eb_lo = add(eb_lo, ld16(rowptr(lat, lw, kyd, kxb_lo, Yd) + Xb0));
        eb_hi = add(eb_hi, ld16(rowptr(lat, lw, kyd, kxb_hi, Yd) + Xb0));
      }
      if (TYPE == PH_FAR) {
        // the other vertical neighbours are ordinary rows; then bring b into a's lane order (lane i <-> i ^ c)
        const int kyd = (ky + 1) & 3, Yd = (Y + (ky == 3)) & Wm;
        ea_lo = add(ea_lo, ld16(rowptr(lat, lw, kyd, 0, Yd) + X0));
        ea_hi = add(ea_hi, ld16(rowptr(lat, lw, kyd, 2, Yd) + X0));
        const int kyu = (kyb - 1) & 3, Yu = (Yb - (kyb == 0)) & Wm;
        eb_lo = add(eb_lo, ld16(rowptr(lat, lw, kyu, kxb_lo, Yu) + Xb0));
        eb_hi = add(eb_hi, ld16(rowptr(lat, lw, kyu, kxb_hi, Yu) + Xb0));
        b_lo = xor_perm<CW>(b_lo, selb); b_hi = xor_perm<CW>(b_hi, selb);
        eb_lo = xor_perm<CW>(eb_lo, selb); eb_hi = xor_perm<CW>(eb_hi, selb);
      } else {
        // vertical domino: a's lower neighbour is b, b's upper neighbour is a
        ea_lo = add(ea_lo, b_lo); ea_hi = add(ea_hi, b_hi);
        eb_lo = add(eb_lo, a_lo); eb_hi = add(eb_hi, a_hi);
      }
      // random words: block c0 = 4*(X>>2) + kx, c1 = y, word X & 3 with X = x>>2, kx = x&3  (U3)
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const u32x4 r0 = philox_update((uint32_t)(4 * (4 * chunk + j) + sel), (uint32_t)y, A.c2, c3, A.key0, A.key1);
        const u32x4 r1 = philox_update((uint32_t)(4 * (4 * chunk + j) + sel + 2), (uint32_t)y, A.c2, c3, A.key0, A.key1);
        process4(a_lo.w[j], b_lo.w[j], ea_lo.w[j], eb_lo.w[j], r0.v[0], r0.v[1], r0.v[2], r0.v[3], s_desc, s_thr, acc);
        process4(a_hi.w[j], b_hi.w[j], ea_hi.w[j], eb_hi.w[j], r1.v[0], r1.v[1], r1.v[2], r1.v[3], s_desc, s_thr, acc);
      }
      if (TYPE == PH_FAR) { b_lo = xor_perm<CW>(b_lo, selb); b_hi = xor_perm<CW>(b_hi, selb); }
      st16(pa_lo, a_lo); st16(pa_hi, a_hi); st16(pb_lo, b_lo); st16(pb_hi, b_hi);
    } else {
      // ---- NEAR, horizontal dominoes: rows ky = half and half + 2 share ka; lanes are indexed by the b-site ------------
      const int ka = (A.p2 + 2 * ((half + A.phase) & 1)) & 3, kb = (ka + 1) & 3;
      const int sh_a = -(ka == 3), sh_l = sh_a - (ka == 0), sh_r = (kb == 3);
      sgn = ((ka + half) & 1) ? -1 : 1;
#pragma unroll
      for (int v = 0; v < 2; ++v) {
        const int ky = half + 2 * v, y = 4 * Y + ky;
        const int kyu = (ky - 1) & 3, Yu = (Y - (ky == 0)) & Wm, kyd = (ky + 1) & 3, Yd = (Y + (ky == 3)) & Wm;
        uint8_t* ra = const_cast<uint8_t*>(rowptr(lat, lw, ky, ka, Y));
        uint8_t* pb = const_cast<uint8_t*>(rowptr(lat, lw, ky, kb, Y)) + X0;
        V16 a = ldrow(ra, X0, W, sh_a), b = ld16(pb);
        V16 ea = add(add(ldrow(rowptr(lat, lw, ky, (ka + 3) & 3, Y), X0, W, sh_l), b),
                     add(ldrow(rowptr(lat, lw, kyu, ka, Yu), X0, W, sh_a), ldrow(rowptr(lat, lw, kyd, ka, Yd), X0, W, sh_a)));
        V16 eb = add(add(a, ldrow(rowptr(lat, lw, ky, (kb + 1) & 3, Y), X0, W, sh_r)),
                     add(ld16(rowptr(lat, lw, kyu, kb, Yu) + X0), ld16(rowptr(lat, lw, kyd, kb, Yd) + X0)));
        // random words, addressed by the b-site: block c0 = 4*(Xb>>2) + kb, c1 = y, word Xb & 3
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const u32x4 rr = philox_update((uint32_t)(4 * (4 * chunk + j) + kb), (uint32_t)y, A.c2, c3, A.key0, A.key1);
          process4(a.w[j], b.w[j], ea.w[j], eb.w[j], rr.v[0], rr.v[1], rr.v[2], rr.v[3], s_desc, s_thr, acc);
        }
        st16(pb, b);
        if (sh_a == 0) st16(ra + X0, a); else st16_left1(ra, X0, W, a);
      }
    }
    // unpack the item's sums: a3 = dJ + (dV << 11) + (dn2 << 22)
    int t = acc.a3;
    const int j11 = (t << 21) >> 21; t = (t - j11) >> 11;
    const int v11 = (t << 21) >> 21; t = (t - v11) >> 11;
    tJ += j11; tV += v11; tn2 += t;
    tM += acc.m16 >> 4;
    tMs += sgn * ((TYPE == PH_FAR ? acc.m16 : acc.d16) >> 4);
  }
  block_accumulate(&A.obs[r], tn2, tV, tJ, tM, tMs);
}

// Public byte codes, row-major  <->  P16 bytes.  One thread per 16 consecutive sites of a row.
__global__ void __launch_bounds__(256) k_codes_to_p16(const int8_t* codes, uint8_t* lat, int logL) {
  const int lw = logL - 2, L = 1 << logL;
  const long long n = ((long long)L * L) >> 4;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(t & ((L >> 4) - 1)), y = (int)(t >> (logL - 4));
    const uint4 v = reinterpret_cast<const uint4*>(codes)[t];
    uint32_t c[4] = {v.x, v.y, v.z, v.w}, e[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) e[k] = (~c[k] & 0x01010101u) | (((c[k] ^ (c[k] >> 1)) & 0x01010101u) << 3);
    const uint32_t t0 = __byte_perm(e[0], e[1], 0x5140), t1 = __byte_perm(e[2], e[3], 0x5140);
    const uint32_t t2 = __byte_perm(e[0], e[1], 0x7362), t3 = __byte_perm(e[2], e[3], 0x7362);
    const uint32_t o[4] = {__byte_perm(t0, t1, 0x5410), __byte_perm(t0, t1, 0x7632), __byte_perm(t2, t3, 0x5410), __byte_perm(t2, t3, 0x7632)};
#pragma unroll
    for (int kx = 0; kx < 4; ++kx)
      *reinterpret_cast<uint32_t*>(lat + p16_site(lw, 16 * j + kx, y)) = o[kx];
  }
}
__global__ void __launch_bounds__(256) k_p16_to_codes(const uint8_t* lat, int8_t* codes, int logL) {
  const int lw = logL - 2, L = 1 << logL;
  const long long n = ((long long)L * L) >> 4;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(t & ((L >> 4) - 1)), y = (int)(t >> (logL - 4));
    uint32_t p[4];
#pragma unroll
    for (int kx = 0; kx < 4; ++kx)
      p[kx] = *reinterpret_cast<const uint32_t*>(lat + p16_site(lw, 16 * j + kx, y));
    const uint32_t t0 = __byte_perm(p[0], p[1], 0x5140), t1 = __byte_perm(p[2], p[3], 0x5140);
    const uint32_t t2 = __byte_perm(p[0], p[1], 0x7362), t3 = __byte_perm(p[2], p[3], 0x7362);
    const uint32_t e[4] = {__byte_perm(t0, t1, 0x5410), __byte_perm(t0, t1, 0x7632), __byte_perm(t2, t3, 0x5410), __byte_perm(t2, t3, 0x7632)};
    uint32_t c[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t b0 = ~e[k] & 0x01010101u;
      c[k] = b0 | ((((e[k] >> 3) ^ b0) & 0x01010101u) << 1);
    }
    reinterpret_cast<uint4*>(codes)[t] = make_uint4(c[0], c[1], c[2], c[3]);
  }
}

// Public byte codes, row-major  <->  P2 words.  One thread per 64 consecutive sites of a row = one word of each of the
// four planes kx.
__global__ void __launch_bounds__(256) k_codes_to_p2(const int8_t* codes, uint8_t* lat, int logL) {
  const int lw = logL - 2, L = 1 << logL;
  const long long n = ((long long)L * L) >> 6;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(t & ((L >> 6) - 1)), y = (int)(t >> (logL - 6));
    V16 pl[4];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const uint4 v = reinterpret_cast<const uint4*>(codes)[4 * t + g];
      uint32_t c[4] = {v.x, v.y, v.z, v.w}, e[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) e[k] = (~c[k] & 0x01010101u) | (((c[k] ^ (c[k] >> 1)) & 0x01010101u) << 3);
      const uint32_t t0 = __byte_perm(e[0], e[1], 0x5140), t1 = __byte_perm(e[2], e[3], 0x5140);
      const uint32_t t2 = __byte_perm(e[0], e[1], 0x7362), t3 = __byte_perm(e[2], e[3], 0x7362);
      pl[0].w[g] = __byte_perm(t0, t1, 0x5410); pl[1].w[g] = __byte_perm(t0, t1, 0x7632);
      pl[2].w[g] = __byte_perm(t2, t3, 0x5410); pl[3].w[g] = __byte_perm(t2, t3, 0x7632);
    }
#pragma unroll
    for (int kx = 0; kx < 4; ++kx)
      *reinterpret_cast<uint32_t*>(lat + p2_word(lw, 64 * j + kx, y)) = pack2(pl[kx]);
  }
}
__global__ void __launch_bounds__(256) k_p2_to_codes(const uint8_t* lat, int8_t* codes, int logL) {
  const int lw = logL - 2, L = 1 << logL;
  const long long n = ((long long)L * L) >> 6;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(t & ((L >> 6) - 1)), y = (int)(t >> (logL - 6));
    V16 pl[4];
#pragma unroll
    for (int kx = 0; kx < 4; ++kx) pl[kx] = widen2(*reinterpret_cast<const uint32_t*>(lat + p2_word(lw, 64 * j + kx, y)));
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const uint32_t p0 = pl[0].w[g], p1 = pl[1].w[g], p2 = pl[2].w[g], p3 = pl[3].w[g];
      const uint32_t t0 = __byte_perm(p0, p1, 0x5140), t1 = __byte_perm(p2, p3, 0x5140);
      const uint32_t t2 = __byte_perm(p0, p1, 0x7362), t3 = __byte_perm(p2, p3, 0x7362);
      const uint32_t e[4] = {__byte_perm(t0, t1, 0x5410), __byte_perm(t0, t1, 0x7632), __byte_perm(t2, t3, 0x5410), __byte_perm(t2, t3, 0x7632)};
      uint32_t c[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t b0 = ~e[k] & 0x01010101u;
        c[k] = b0 | ((((e[k] >> 3) ^ b0) & 0x01010101u) << 1);
      }
      reinterpret_cast<uint4*>(codes)[4 * t + g] = make_uint4(c[0], c[1], c[2], c[3]);
    }
  }
}

// Full recomputation of (n2, bV, bJ, M, Ms, Q) from eq. (3) on the tiled layout: one thread per 16-byte
// plane vector, bit logic on the (f, g) bytes.  A site is a charge iff f == g (S = f + g - 1), else a spin (sigma = f - g);
// for a bond (i, j): S_i S_j = +-1 iff both are charges (sign: f_i == f_j), sigma_i sigma_j = +-1 iff both are spins.
// Every site owns its +x and +y bond: the +x neighbour of plane kx is plane kx+1 (plane 0 one column on for kx = 3), the
// +y neighbour of row ky is row ky+1 (row 0 of the next quad for ky = 3).  out8 must be zeroed before the launch.
template <int BITS>
__global__ void __launch_bounds__(256) k_recompute_p16(const uint8_t* lat, int logL, long long* out8) {
  const int lw = logL - 2, W = 1 << lw, ls = p16_logseg(lw), SEGL = 1 << ls;
  const long long nvec = ((long long)1 << (2 * logL)) >> 4;
  long long acc[6] = {0, 0, 0, 0, 0, 0};
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < nvec; t += (long long)gridDim.x * blockDim.x) {
    // t = ((Y * 16 + row) * (W / 16)) + chunk
    const int chunk = (int)(t & ((W >> 4) - 1));
    const int row = (int)(t >> (lw - 4)) & 15, Y = (int)(t >> lw);
    const int ky = row >> 2, kx = row & 3, X0 = chunk << 4;
    const int seg = X0 >> ls, xo = X0 & (SEGL - 1);
    const V16 v = ldvec<BITS>(lat, p16_row(lw, ky, kx, Y, seg) + xo);
    V16 rgt;
    if (kx < 3) rgt = ldvec<BITS>(lat, p16_row(lw, ky, kx + 1, Y, seg) + xo);
    else {
      const int Xn = (X0 + 16) & (W - 1);
      rgt = shift_down(ldvec<BITS>(lat, p16_row(lw, ky, 0, Y, seg) + xo), ldsite<BITS>(lat, p16_row(lw, ky, 0, Y, Xn >> ls) + (Xn & (SEGL - 1))));
    }
    const V16 dwn = ky < 3 ? ldvec<BITS>(lat, p16_row(lw, ky + 1, kx, Y, seg) + xo) : ldvec<BITS>(lat, p16_row(lw, 0, kx, (Y + 1) & (W - 1), seg) + xo);
    int n2 = 0, bV = 0, bJ = 0, nf = 0, ng = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t m = 0x01010101u;
      const uint32_t f = v.w[k] & m, g = (v.w[k] >> 3) & m, ch = ~(f ^ g) & m;
      nf += __popc(f); ng += __popc(g); n2 += __popc(ch);
#pragma unroll
      for (int dir = 0; dir < 2; ++dir) {
        const uint32_t u = dir ? dwn.w[k] : rgt.w[k];
        const uint32_t fu = u & m, gu = (u >> 3) & m, chu = ~(fu ^ gu) & m, same = ~(f ^ fu) & m;
        const uint32_t cc = ch & chu, ss = ~ch & ~chu & m;
        bV += __popc(cc & same) - __popc(cc & ~same);
        bJ += __popc(ss & same) - __popc(ss & ~same);
      }
    }
    const int Mv = nf - ng;
    acc[0] += n2; acc[1] += bV; acc[2] += bJ; acc[3] += Mv; acc[4] += ((kx + ky) & 1) ? -Mv : Mv; acc[5] += nf + ng - 16;
  }
  __shared__ long long red[6][8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    long long q = acc[k];
    for (int o = 16; o > 0; o >>= 1) q += __shfl_down_sync(0xFFFFFFFFu, q, o);
    if (lane == 0) red[k][warp] = q;
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    long long q = 0;
    for (int wv = 0; wv < 8; ++wv) q += red[threadIdx.x][wv];
    atomicAdd((unsigned long long*)&out8[threadIdx.x], (unsigned long long)q);
  }
}

// Validation of a lattice in public byte codes (ic_set_state): out2[0] = number of bytes outside 0..3, out2[1] = sum S.
__global__ void __launch_bounds__(256) k_validate_codes(const int8_t* codes, long long n16, long long* out2) {
  long long bad = 0, q = 0;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n16; t += (long long)gridDim.x * blockDim.x) {
    const uint4 v = reinterpret_cast<const uint4*>(codes)[t];
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      bad += (w[k] & 0xFCFCFCFCu) != 0u;
      const uint32_t ch = (w[k] >> 1) & 0x01010101u;          // bit1 = charge, bit0 = negative
      q += __popc(ch) - 2 * __popc(ch & w[k]);
    }
  }
  for (int o = 16; o > 0; o >>= 1) { bad += __shfl_down_sync(0xFFFFFFFFu, bad, o); q += __shfl_down_sync(0xFFFFFFFFu, q, o); }
  if ((threadIdx.x & 31) == 0) {
    if (bad) atomicAdd((unsigned long long*)&out2[0], (unsigned long long)bad);
    if (q) atomicAdd((unsigned long long*)&out2[1], (unsigned long long)q);
  }
}

}  // namespace ic
