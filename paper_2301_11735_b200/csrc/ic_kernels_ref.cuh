// ic_kernels_ref.cuh -- variant 1: one thread per coupled pair, lattice in global memory.
//
// The plain CUDA statement of the pair update (sec. 3.1) under schedule S1 (U4).
// It runs any power-of-two L >= 4 in every layout (ROW8, ROW2, P16) and is the in-library cross-check for the
// tiled kernels; it is also what small lattices (L < 64) and 2-bit states use.  Each thread recomputes the Philox block
// of its group of four pairs and keeps one word.
#pragma once
#include "ic_common.cuh"

namespace ic {

// Sum of five per-thread integers over the block, then one atomicAdd per value into the replica record.
// absolute = false: dM, dMs are changes of M, Ms; true: they are the M, Ms of the sites updated (added to Mnext, Msnext).
__device__ __forceinline__ void block_accumulate(ReplicaObs* o, int dn2, int dV, int dJ, int dM, int dMs, bool absolute = false) {
  __shared__ int red[5][32];
  const unsigned full = 0xFFFFFFFFu;
  dn2 = __reduce_add_sync(full, dn2); dV = __reduce_add_sync(full, dV); dJ = __reduce_add_sync(full, dJ);
  dM = __reduce_add_sync(full, dM); dMs = __reduce_add_sync(full, dMs);
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
  if (lane == 0) { red[0][warp] = dn2; red[1][warp] = dV; red[2][warp] = dJ; red[3][warp] = dM; red[4][warp] = dMs; }
  __syncthreads();
  if (warp == 0) {
    int v[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) v[k] = __reduce_add_sync(full, lane < nwarp ? red[k][lane] : 0);
    if (lane == 0) {
      if (v[0]) atomicAdd((unsigned long long*)&o->n2, (unsigned long long)(long long)v[0]);
      if (v[1]) atomicAdd((unsigned long long*)&o->bV, (unsigned long long)(long long)v[1]);
      if (v[2]) atomicAdd((unsigned long long*)&o->bJ, (unsigned long long)(long long)v[2]);
      if (v[3]) atomicAdd((unsigned long long*)(absolute ? &o->Mnext : &o->M), (unsigned long long)(long long)v[3]);
      if (v[4]) atomicAdd((unsigned long long*)(absolute ? &o->Msnext : &o->Ms), (unsigned long long)(long long)v[4]);
    }
  }
}

// Lattice accessors for the pair update below: global memory in any layout, or a row-major byte lattice in shared memory.
template <int LAY>
struct GlobalLat {
  LatView v;
  __device__ __forceinline__ int load(int x, int y) const { return Sites<LAY>::load(v, x, y); }
  __device__ __forceinline__ void store(int x, int y, int oldc, int newc) const { Sites<LAY>::store(v, x, y, oldc, newc); }
};
struct SmemLat {
  int8_t* s; int logL;
  __device__ __forceinline__ int load(int x, int y) const { return s[(y << logL) + x]; }
  __device__ __forceinline__ void store(int x, int y, int, int newc) const { s[(y << logL) + x] = (int8_t)newc; }
};

// One coupled-pair update of the pair a = (xa, ya), b = (xb, yb) with the random word w, adj = 1 if b is a
// neighbour of a (eq. 5) else 0 (eq. 4).  thr(class) returns 8*t29 - 1 of the replica.  Adds the accepted move's changes to
// dn2, dV, dJ, dM, dMs.
template <class Lat, class Thr>
__device__ __forceinline__ void pair_update_core(const Lat& lat, int L, int xa, int ya, int xb, int yb, int adj, uint32_t w, const Thr& thr,
                                                 int& dn2, int& dV, int& dJ, int& dM, int& dMs) {
  const int mask = L - 1;
  // --- proposal: same pair charge q, configuration r of the paper's list ----------
  // all ten sites are loaded up front (independent loads: one memory latency instead of three in a row)
  const int ca = lat.load(xa, ya), cb = lat.load(xb, yb);
  const int xl = (xa - 1) & mask, xr = (xa + 1) & mask, yu = (ya - 1) & mask, yd = (ya + 1) & mask;
  const int a1 = lat.load(xl, ya), a2 = lat.load(xr, ya);
  const int a3 = lat.load(xa, yu), a4 = lat.load(xa, yd);
  const int xl2 = (xb - 1) & mask, xr2 = (xb + 1) & mask, yu2 = (yb - 1) & mask, yd2 = (yb + 1) & mask;
  const int e1 = lat.load(xl2, yb), e2 = lat.load(xr2, yb);
  const int e3 = lat.load(xb, yu2), e4 = lat.load(xb, yd2);
  const int q = S_of(ca) + S_of(cb);
  const int rr = (int)(w & 7u);
  int na = ca, nb = cb;
  if (q == 0) {
    // (S+,S-) (S-,S+) (s+,s+) (s-,s-) (s+,s-) (s-,s+); rr = 6,7: nothing proposed
    switch (rr) {
      case 0: na = 2; nb = 3; break;
      case 1: na = 3; nb = 2; break;
      case 2: na = 0; nb = 0; break;
      case 3: na = 1; nb = 1; break;
      case 4: na = 0; nb = 1; break;
      case 5: na = 1; nb = 0; break;
      default: na = ca; nb = cb; break;
    }
  } else if (q == 1 || q == -1) {
    const int C = q > 0 ? 2 : 3;     // (C,s+) (C,s-) (s+,C) (s-,C)
    switch (rr & 3) {
      case 0: na = C; nb = 0; break;
      case 1: na = C; nb = 1; break;
      case 2: na = 0; nb = C; break;
      default: na = 1; nb = C; break;
    }
  }
  if (na != ca || nb != cb) {
    // --- neighbour sums over the four slots of a and of b, current lattice ----------
    const int nSa = S_of(a1) + S_of(a2) + S_of(a3) + S_of(a4), nGa = sg_of(a1) + sg_of(a2) + sg_of(a3) + sg_of(a4);
    const int nSb = S_of(e1) + S_of(e2) + S_of(e3) + S_of(e4), nGb = sg_of(e1) + sg_of(e2) + sg_of(e3) + sg_of(e4);
    // --- dE class: eq. (4) distant / eq. (5) neighbouring sites, spin term as in DESIGN.md G1 ------
    const int dSa = S_of(na) - S_of(ca), dSb = S_of(nb) - S_of(cb);
    const int dGa = sg_of(na) - sg_of(ca), dGb = sg_of(nb) - sg_of(cb);
    const int e_d = S_of(na) * S_of(na) + S_of(nb) * S_of(nb) - S_of(ca) * S_of(ca) - S_of(cb) * S_of(cb);
    const int e_v = dSa * nSa + dSb * nSb + adj * dSa * dSb;
    const int e_j = dGa * nGa + dGb * nGb + adj * dGa * dGb;
    const uint32_t t8 = thr(class_index(e_d, e_v, e_j));
    if (w <= t8) {                   // Metropolis min(1, exp(-dE/T)): (w >> 3) < t29, t8 = 8 t29 - 1
      lat.store(xa, ya, ca, na);
      lat.store(xb, yb, cb, nb);
      dn2 += e_d; dV += e_v; dJ += e_j; dM += dGa + dGb;
      dMs += (((xa + ya) & 1) ? -dGa : dGa) + (((xb + yb) & 1) ? -dGb : dGb);
    }
  }
}

// The t-th coupled pair of a phase of schedule S1 (U4), updated as the paper states it:
// the plain CUDA statement of the method.  thr(class) returns 8*t29 - 1 of the replica.  Adds the accepted move's
// changes to dn2, dV, dJ, dM, dMs.
template <class Lat, class Thr>
__device__ __forceinline__ void ref_pair_update(const Lat& lat, int L, int logL, int type, int p1, int p2, int phase, uint32_t c2,
                                                uint32_t c3, uint32_t key0, uint32_t key1, const Thr& thr, long long t,
                                                int& dn2, int& dV, int& dJ, int& dM, int& dMs) {
  const int mask = L - 1;
  // --- which pair (schedule S1) and which random word ---------------------------------------------
  int xa, ya, xb, yb, adj; uint32_t c0, word;
  if (type == 0) {                 // FAR: a = (even x, y = phase mod 2), b = (x^mx, y^my); eq. (4)
    int i = (int)(t & ((L >> 1) - 1)), j = (int)(t >> (logL - 1));
    xa = 2 * i; ya = 2 * j + phase; xb = xa ^ p1; yb = ya ^ p2; adj = 0;
    c0 = (((uint32_t)xa >> 4) << 2) | ((uint32_t)xa & 3u); word = ((uint32_t)xa >> 2) & 3u;
  } else if (p1 == 0) {            // NEAR, horizontal dominoes (brick pattern); eq. (5)
    int i = (int)(t & ((L >> 2) - 1)); ya = (int)(t >> (logL - 2));
    xa = ((p2 + 2 * ((ya + phase) & 1)) & 3) + 4 * i; xb = (xa + 1) & mask; yb = ya; adj = 1;
    c0 = (((uint32_t)xb >> 4) << 2) | ((uint32_t)xb & 3u); word = ((uint32_t)xb >> 2) & 3u;   // addressed by the b-site
  } else {                           // NEAR, vertical dominoes
    xa = (int)(t & mask); int jy = (int)(t >> logL);
    ya = ((p2 + 2 * ((xa + phase) & 1)) & 3) + 4 * jy; xb = xa; yb = (ya + 1) & mask; adj = 1;
    c0 = (((uint32_t)xa >> 4) << 2) | ((uint32_t)xa & 3u); word = ((uint32_t)xa >> 2) & 3u;
  }
  u32x4 rnd = philox_update(c0, (uint32_t)ya, c2, c3, key0, key1);
  uint32_t w = word == 0 ? rnd.v[0] : word == 1 ? rnd.v[1] : word == 2 ? rnd.v[2] : rnd.v[3];
  pair_update_core(lat, L, xa, ya, xb, yb, adj, w, thr, dn2, dV, dJ, dM, dMs);
}

template <int LAY>
__global__ void __launch_bounds__(256) k_ref_phase(PhaseArgs A) {
  asm volatile("griddepcontrol.launch_dependents;");      // programmatic dependent launch: see launch_pdl (ic_api.cu)
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int L = A.L, logL = A.logL;
  const int r = blockIdx.y;
  const long long npairs = ((long long)L * L) >> 2;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const GlobalLat<LAY> lat{LatView{(char*)A.lattice + (long long)r * A.lat_stride, L, logL}};
  const uint2* thr_r = A.thr + (long long)r * THR_STRIDE;
  auto thr = [thr_r](int cls) -> uint32_t { return __ldg(&thr_r[cls]).x; };
  int dn2 = 0, dV = 0, dJ = 0, dM = 0, dMs = 0;
  if (t < npairs)
    ref_pair_update(lat, L, logL, A.type, A.p1, A.p2, A.phase, A.c2, (uint32_t)r | (TAG_UPDATE << 28), A.key0, A.key1, thr, t,
                    dn2, dV, dJ, dM, dMs);
  block_accumulate(&A.obs[r], dn2, dV, dJ, dM, dMs);
}

// U5: after a sweep, E = Delta*n2 + V*bV + (J/4)*bJ and the running sums, one thread per
// replica, IEEE fp64 with one rounding per operation (no FMA contraction: explicit _rn intrinsics).
__global__ void k_fold(ReplicaObs* obs, int replicas, double delta, double V, double quarterJ, long long* trace_row, int absolute,
                       unsigned int* task_ctr) {
  asm volatile("griddepcontrol.launch_dependents;");   // no-ops unless launched as a programmatic dependent (staged path)
  asm volatile("griddepcontrol.wait;" ::: "memory");
  int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= replicas) return;
  ReplicaObs* o = &obs[r];
  if (task_ctr) { task_ctr[TASK_CTR_STRIDE * r] = 0u; task_ctr[TASK_CTR_STRIDE * r + 1] = 0u; }   // both phases are complete: the staged kernels' task counters
  if (absolute) { o->M = o->Mnext; o->Ms = o->Msnext; o->Mnext = 0; o->Msnext = 0; }   // the two phases covered every site once
  const double E = __dadd_rn(__dadd_rn(__dmul_rn(delta, (double)o->n2), __dmul_rn(V, (double)o->bV)),
                             __dmul_rn(quarterJ, (double)o->bJ));
  const double M = (double)o->M, Ms = (double)o->Ms;
  o->sumE = __dadd_rn(o->sumE, E); o->sumE2 = __dadd_rn(o->sumE2, __dmul_rn(E, E));
  o->sumM = __dadd_rn(o->sumM, M); o->sumM2 = __dadd_rn(o->sumM2, __dmul_rn(M, M)); o->sumAbsM = __dadd_rn(o->sumAbsM, fabs(M));
  o->sumMs = __dadd_rn(o->sumMs, Ms); o->sumMs2 = __dadd_rn(o->sumMs2, __dmul_rn(Ms, Ms)); o->sumAbsMs = __dadd_rn(o->sumAbsMs, fabs(Ms));
  o->nmeas += 1;
  if (trace_row) {
    long long* t = trace_row + 6LL * r;
    t[0] = o->n2; t[1] = o->bV; t[2] = o->bJ; t[3] = o->M; t[4] = o->Ms; t[5] = o->Q;
  }
}

// Full recomputation of (n2, bV, bJ, M, Ms, Q) straight from eq. (3): every site contributes
// its on-site term and its +x and +y bond, periodic.  out8 must be zeroed before the launch.
template <int LAY>
__global__ void __launch_bounds__(256) k_recompute(LatView lat, long long* out8) {
  const int L = lat.L, logL = lat.logL;
  const long long N = (long long)L * L;
  const int mask = L - 1;
  long long acc[6] = {0, 0, 0, 0, 0, 0};
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    const int x = (int)(i & mask), y = (int)(i >> logL);
    const int c = Sites<LAY>::load(lat, x, y);
    const int cr = Sites<LAY>::load(lat, (x + 1) & mask, y);
    const int cd = Sites<LAY>::load(lat, x, (y + 1) & mask);
    const int S = S_of(c), G = sg_of(c);
    acc[0] += S * S; acc[1] += S * (S_of(cr) + S_of(cd)); acc[2] += G * (sg_of(cr) + sg_of(cd));
    acc[3] += G; acc[4] += ((x + y) & 1) ? -G : G; acc[5] += S;
  }
  __shared__ long long red[6][8];
  int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 6; ++k) {
    long long v = acc[k];
    for (int s = 16; s > 0; s >>= 1) v += __shfl_down_sync(0xFFFFFFFFu, v, s);
    if (lane == 0) red[k][warp] = v;
  }
  __syncthreads();
  if (threadIdx.x < 6) {
    long long v = 0;
    for (int wv = 0; wv < (int)(blockDim.x >> 5); ++wv) v += red[threadIdx.x][wv];
    atomicAdd((unsigned long long*)&out8[threadIdx.x], (unsigned long long)v);
  }
}

// Public byte codes <-> 2-bit packed words (16 sites per word).  n16 = number of words.
__global__ void k_pack2(const int8_t* codes, uint32_t* words, long long n16) {
  for (long long wi = (long long)blockIdx.x * blockDim.x + threadIdx.x; wi < n16; wi += (long long)gridDim.x * blockDim.x) {
    const uint4 v = ((const uint4*)codes)[wi];
    const uint32_t in[4] = {v.x, v.y, v.z, v.w};
    uint32_t out = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      uint32_t b = in[k] & 0x03030303u;                       // four codes, one per byte
      b = (b | (b >> 6)) & 0x000F000Fu; b = (b | (b >> 12)) & 0xFFu;  // -> 8 bits
      out |= b << (8 * k);
    }
    words[wi] = out;
  }
}
__global__ void k_unpack2(const uint32_t* words, int8_t* codes, long long n16) {
  for (long long wi = (long long)blockIdx.x * blockDim.x + threadIdx.x; wi < n16; wi += (long long)gridDim.x * blockDim.x) {
    const uint32_t wd = words[wi];
    uint32_t out[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      uint32_t b = (wd >> (8 * k)) & 0xFFu;
      b = (b | (b << 12)) & 0x000F000Fu; b = (b | (b << 6)) & 0x03030303u;
      out[k] = b;
    }
    ((uint4*)codes)[wi] = make_uint4(out[0], out[1], out[2], out[3]);
  }
}

// Sum S of a lattice in packed public codes (ic_set_state_packed): every 2-bit pattern is a valid code, so eq. (2)
// is the only thing to check.  code bit1 = charge, bit0 = negative.  out2[1] += sum S.
__global__ void __launch_bounds__(256) k_charge_of_packed(const uint32_t* words, long long n16, long long* out2) {
  long long q = 0;
  for (long long wi = (long long)blockIdx.x * blockDim.x + threadIdx.x; wi < n16; wi += (long long)gridDim.x * blockDim.x) {
    const uint32_t wd = words[wi], ch = (wd >> 1) & 0x55555555u;
    q += __popc(ch) - 2 * __popc(ch & wd);
  }
  for (int o = 16; o > 0; o >>= 1) q += __shfl_down_sync(0xFFFFFFFFu, q, o);
  if ((threadIdx.x & 31) == 0 && q) atomicAdd((unsigned long long*)&out2[1], (unsigned long long)q);
}

}  // namespace ic
