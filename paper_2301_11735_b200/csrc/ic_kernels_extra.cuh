// ic_kernels_extra.cuh -- what the paper describes around its main algorithm, on the device:
//
//   * maps: a map is a list of coupled pairs that do not interact; the paper builds maps of N/10 pairs
//     on the CPU (sequential rejection sampling over an L x L bool array) and ships them over PCIe.
//     Here a map is built on the device in one round: K candidate pairs of two distinct uniformly random sites from the
//     counter-based stream; candidate k survives iff no candidate of lower index has a site inside its covering (its two
//     sites and their nearest neighbours, Fig. 1).  Survivors are mutually non-interacting by construction.
//     Then one thread per surviving pair and lattice copy does the coupled-pair update, the same map for
//     every copy.
//   * the largest connected cluster of charged sites, the "drop" of PAPER.md:161-163 (Fig. 7): union-find over the
//     charged sites with atomicMin links, 4-neighbour connectivity, periodic.
#pragma once
#include "ic_common.cuh"
#include "ic_kernels_ref.cuh"

namespace ic {

enum : uint32_t { TAG_MAP = 6, TAG_MAPU = 7 };

struct MapArgs {
  void* lattice; const uint2* thr; ReplicaObs* obs;
  int* first;                  // [N]: lowest index of a candidate with this site (K if none)
  int* ia; int* ib;            // [K] candidate sites
  long long lat_stride;
  int L, logL, K, replicas;
  uint32_t map_index, key0, key1;
};

__global__ void k_map_reset(int* first, long long N, int K) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) first[i] = K;
}

// candidate k: a = (w0 N) >> 32, b = (w1 (N-1)) >> 32 skipping a, words of Philox4x32-10(ctr = (k, 0, map, MAP))
__global__ void k_map_candidates(MapArgs A) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= A.K) return;
  const unsigned long long N = 1ull << (2 * A.logL);
  const u32x4 w = philox4x32_10((uint32_t)k, 0u, A.map_index, TAG_MAP << 28, A.key0, A.key1);
  const int a = (int)(((unsigned long long)w.v[0] * N) >> 32);
  int b = (int)(((unsigned long long)w.v[1] * (N - 1)) >> 32);
  if (b >= a) ++b;
  A.ia[k] = a; A.ib[k] = b;
  atomicMin(&A.first[a], k); atomicMin(&A.first[b], k);
}

// one thread per (candidate, replica): survival test, then the coupled-pair update of PAPER.md:64-98
template <int LAY>
__global__ void __launch_bounds__(256) k_map_update(MapArgs A) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x, r = blockIdx.y;
  int dn2 = 0, dV = 0, dJ = 0, dM = 0, dMs = 0;
  if (k < A.K) {
    const int L = A.L, mask = L - 1, a = A.ia[k], b = A.ib[k];
    const int xa = a & mask, ya = a >> A.logL, xb = b & mask, yb = b >> A.logL;
    bool alive = true;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int x = e ? xb : xa, y = e ? yb : ya;
      alive = alive && A.first[(y << A.logL) + x] >= k && A.first[(y << A.logL) + ((x + 1) & mask)] >= k &&
              A.first[(y << A.logL) + ((x - 1) & mask)] >= k && A.first[(((y + 1) & mask) << A.logL) + x] >= k &&
              A.first[(((y - 1) & mask) << A.logL) + x] >= k;
    }
    if (alive) {
      const int adj = (ya == yb && (((xa + 1) & mask) == xb || ((xa - 1) & mask) == xb)) ||
                      (xa == xb && (((ya + 1) & mask) == yb || ((ya - 1) & mask) == yb)) ? 1 : 0;
      const u32x4 w = philox4x32_10((uint32_t)(k >> 2), 1u, A.map_index, (uint32_t)r | (TAG_MAPU << 28), A.key0, A.key1);
      const uint32_t word = (k & 3) == 0 ? w.v[0] : (k & 3) == 1 ? w.v[1] : (k & 3) == 2 ? w.v[2] : w.v[3];
      const GlobalLat<LAY> lat{LatView{(char*)A.lattice + (long long)r * A.lat_stride, L, A.logL}};
      const uint2* thr_r = A.thr + (long long)r * THR_STRIDE;
      auto thr = [thr_r](int cls) -> uint32_t { return __ldg(&thr_r[cls]).x; };
      pair_update_core(lat, L, xa, ya, xb, yb, adj, word, thr, dn2, dV, dJ, dM, dMs);
    }
  }
  block_accumulate(&A.obs[r], dn2, dV, dJ, dM, dMs);
}

// ---------------------------------------------------------------------------------------------------------------
// Largest cluster of charged sites.  which: 0 S != 0, 1 S = +1, 2 S = -1.  parent[i] = i for sites inside, -1 outside.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool cc_inside(int c, int which) { return which == 0 ? c >= 2 : which == 1 ? c == 2 : c == 3; }

template <int LAY>
__global__ void k_cc_init(LatView lat, int which, int* parent, int* size) {
  const long long N = (long long)lat.L * lat.L;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    const int c = Sites<LAY>::load(lat, (int)(i & (lat.L - 1)), (int)(i >> lat.logL));
    parent[i] = cc_inside(c, which) ? (int)i : -1;
    size[i] = 0;
  }
}
__device__ __forceinline__ int cc_find(const int* parent, int i) {
  int p = ((volatile const int*)parent)[i];
  while (p != i) { i = p; p = ((volatile const int*)parent)[i]; }
  return i;
}
__device__ __forceinline__ void cc_union(int* parent, int a, int b) {
  while (true) {
    a = cc_find(parent, a); b = cc_find(parent, b);
    if (a == b) return;
    if (a < b) { const int t = a; a = b; b = t; }          // link the larger root under the smaller
    const int old = atomicMin(&parent[a], b);
    if (old == a) return;
    a = old;
  }
}
__global__ void k_cc_link(int L, int logL, int* parent) {
  const long long N = (long long)L * L;
  const int mask = L - 1;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    if (parent[i] < 0) continue;
    const int x = (int)(i & mask), y = (int)(i >> logL);
    const int jr = (y << logL) + ((x + 1) & mask), jd = (((y + 1) & mask) << logL) + x;
    if (jr != (int)i && ((volatile int*)parent)[jr] >= 0) cc_union(parent, (int)i, jr);
    if (jd != (int)i && ((volatile int*)parent)[jd] >= 0) cc_union(parent, (int)i, jd);
  }
}
__global__ void k_cc_count(long long N, const int* parent, int* size) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x)
    if (parent[i] >= 0) atomicAdd(&size[cc_find(parent, (int)i)], 1);
}
// out2[0] = largest size, out2[1] = number of clusters (both zeroed before the launch)
__global__ void k_cc_max(long long N, const int* size, long long* out2) {
  long long best = 0, n = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    const int s = size[i];
    if (s > 0) { ++n; if (s > best) best = s; }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const long long ob = __shfl_down_sync(0xFFFFFFFFu, best, o), on = __shfl_down_sync(0xFFFFFFFFu, n, o);
    best = ob > best ? ob : best; n += on;
  }
  if ((threadIdx.x & 31) == 0) {
    if (best) atomicMax((unsigned long long*)&out2[0], (unsigned long long)best);
    if (n) atomicAdd((unsigned long long*)&out2[1], (unsigned long long)n);
  }
}

}  // namespace ic
