// ic_kernels_resident.cuh -- variant 4: small lattices (L <= 64, configs C1 and C2 of BASELINE.json).
//
// A sweep of a 16 x 16 or 64 x 64 lattice is a few hundred to a few thousand pair updates: launching two phase kernels
// and a fold per sweep makes such runs launch-bound.  Here ONE launch runs all the sweeps of an ic_sweep call: one block
// per replica keeps the replica's lattice (public codes, one byte per site) and its threshold table in shared memory,
// derives the schedule of every sweep itself (the same Philox call the host would make, U4), separates the two
// phases by __syncthreads, reduces the observables' changes over the block and lets thread 0 do the per-sweep fold
// (U5, the operations of k_fold in the same order).  The pair update is ref_pair_update (ic_kernels_ref.cuh), the plain
// statement of PAPER.md:64-98; random-number addresses are those of every other kernel, so lattices are identical.
#pragma once
#include "ic_common.cuh"
#include "ic_kernels_ref.cuh"

namespace ic {

constexpr int RES_MAX_L = 64;
constexpr int RES_THREADS = 512;           // at most; the host launches one thread per pair of a phase, 64 <= threads <= 512

struct ResidentArgs {
  void* lattice;                 // [replicas][lat_stride bytes]
  const uint2* thr;              // [replicas][THR_STRIDE]
  ReplicaObs* obs;               // [replicas]
  long long* trace;              // nullptr or [nsweeps][replicas][6]
  long long lat_stride;
  long long nsweeps;
  unsigned long long sweep0;     // global index of the first sweep
  double delta, V, quarterJ;
  int L, logL, replicas;
  uint32_t key0, key1;
};

template <int LAY>
__global__ void __launch_bounds__(RES_THREADS) k_resident_sweeps(ResidentArgs A) {
  __shared__ int8_t s_code[RES_MAX_L * RES_MAX_L];
  __shared__ uint32_t s_thr[THR_STRIDE];
  __shared__ int s_par[4];
  __shared__ int s_red[5][RES_THREADS / 32];
  const int r = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int L = A.L, logL = A.logL, N = L * L, npairs = N >> 2;
  const LatView gv{(char*)A.lattice + (long long)r * A.lat_stride, L, logL};
  const int nthr = (int)blockDim.x;
  for (int k = tid; k < THR_STRIDE; k += nthr) s_thr[k] = __ldg(&A.thr[(long long)r * THR_STRIDE + k]).x;
  for (int i = tid; i < N; i += nthr) s_code[i] = (int8_t)Sites<LAY>::load(gv, i & (L - 1), i >> logL);
  ReplicaObs o;
  if (tid == 0) o = A.obs[r];
  const SmemLat lat{s_code, logL};
  auto thr = [&](int cls) -> uint32_t { return s_thr[cls]; };
  const uint32_t c3 = (uint32_t)r | (TAG_UPDATE << 28);
  __syncthreads();

  for (long long s = 0; s < A.nsweeps; ++s) {
    const unsigned long long sweep = A.sweep0 + (unsigned long long)s;
    if (tid == 0) {
      // U4: parameters of the sweep, the same for all replicas (identical maps for all copies)
      const u32x4 z = philox4x32_10(0u, 0u, (uint32_t)sweep, TAG_SCHED << 28, A.key0, A.key1);
      if ((sweep & 1) == 0) { s_par[0] = 0; s_par[1] = (int)(2 * (z.v[0] & (uint32_t)(L / 2 - 1)) + 1); s_par[2] = (int)(2 * (z.v[1] & (uint32_t)(L / 2 - 1)) + 1); }
      else { s_par[0] = 1; s_par[1] = (int)(z.v[0] & 1u); s_par[2] = (int)(z.v[1] & 3u); }
    }
    __syncthreads();
    const int type = s_par[0], p1 = s_par[1], p2 = s_par[2];
    int dn2 = 0, dV = 0, dJ = 0, dM = 0, dMs = 0;
    for (int phase = 0; phase < 2; ++phase) {
      const uint32_t c2 = (uint32_t)(2 * sweep + (unsigned long long)phase);
      for (int t = tid; t < npairs; t += nthr)
        ref_pair_update(lat, L, logL, type, p1, p2, phase, c2, c3, A.key0, A.key1, thr, (long long)t, dn2, dV, dJ, dM, dMs);
      __syncthreads();       // phase 1 reads neighbours written in phase 0
    }
    const unsigned full = 0xFFFFFFFFu;
    dn2 = __reduce_add_sync(full, dn2); dV = __reduce_add_sync(full, dV); dJ = __reduce_add_sync(full, dJ);
    dM = __reduce_add_sync(full, dM); dMs = __reduce_add_sync(full, dMs);
    if (lane == 0) { s_red[0][warp] = dn2; s_red[1][warp] = dV; s_red[2][warp] = dJ; s_red[3][warp] = dM; s_red[4][warp] = dMs; }
    __syncthreads();
    if (tid == 0) {
      for (int wv = 0; wv < (nthr >> 5); ++wv) {
        o.n2 += s_red[0][wv]; o.bV += s_red[1][wv]; o.bJ += s_red[2][wv]; o.M += s_red[3][wv]; o.Ms += s_red[4][wv];
      }
      // U5, one rounding per operation, the order of k_fold
      const double E = __dadd_rn(__dadd_rn(__dmul_rn(A.delta, (double)o.n2), __dmul_rn(A.V, (double)o.bV)),
                                 __dmul_rn(A.quarterJ, (double)o.bJ));
      const double M = (double)o.M, Ms = (double)o.Ms;
      o.sumE = __dadd_rn(o.sumE, E); o.sumE2 = __dadd_rn(o.sumE2, __dmul_rn(E, E));
      o.sumM = __dadd_rn(o.sumM, M); o.sumM2 = __dadd_rn(o.sumM2, __dmul_rn(M, M)); o.sumAbsM = __dadd_rn(o.sumAbsM, fabs(M));
      o.sumMs = __dadd_rn(o.sumMs, Ms); o.sumMs2 = __dadd_rn(o.sumMs2, __dmul_rn(Ms, Ms)); o.sumAbsMs = __dadd_rn(o.sumAbsMs, fabs(Ms));
      o.nmeas += 1;
      if (A.trace) {
        long long* tr = A.trace + 6LL * ((long long)A.replicas * s + r);
        tr[0] = o.n2; tr[1] = o.bV; tr[2] = o.bJ; tr[3] = o.M; tr[4] = o.Ms; tr[5] = o.Q;
      }
    }
    // s_red is rewritten only after the three barriers of the next sweep
  }
  __syncthreads();
  // write the lattice back in its layout
  if (LAY == LAY_ROW2) {
    uint32_t* words = reinterpret_cast<uint32_t*>(gv.base);
    for (int wi = tid; wi < (N >> 4); wi += nthr) {
      uint32_t wd = 0;
#pragma unroll
      for (int k = 0; k < 16; ++k) wd |= (uint32_t)(s_code[16 * wi + k] & 3) << (2 * k);
      words[wi] = wd;
    }
  } else {
    for (int i = tid; i < N; i += nthr) Sites<LAY>::store(gv, i & (L - 1), i >> logL, 0, s_code[i]);
  }
  if (tid == 0) A.obs[r] = o;
}

}  // namespace ic
