// ic_api.cu -- host side of libic_b200: the C ABI of include/ic.h.
//
// Validates arguments, carves the caller's workspace, builds the acceptance-threshold tables (U2) and the
// O(1) schedule parameters of each sweep (U4), and launches the sm_100a kernels.  No lattice arithmetic runs
// on the host except stage 1 of the algorithm (the initial configuration with the prescribed
// charge), which is a sequential selection and belongs to ic_create, not to the sweep.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "../../include/ic.h"
#include "ic_common.cuh"
#include "ic_kernels_ref.cuh"
#include "ic_kernels_p16.cuh"
#include "ic_kernels_staged.cuh"
#include "ic_kernels_resident.cuh"
#include "ic_kernels_coop.cuh"
#include "ic_kernels_extra.cuh"

using namespace ic;

struct ic_ctx {
  int L, logL, replicas, bits, variant, layout;
  long long N, Q;
  double n, delta, V, J;
  uint64_t seed, sweep;
  cudaStream_t stream;
  // device (inside the caller's workspace)
  char* lattice; long long lat_stride;
  uint2* d_thr; uint2* d_desc; uint2* d_desc32; ReplicaObs* d_obs; long long* d_scratch8; CoopScratch* d_coop; unsigned int* d_task_ctr; int8_t* d_stage; uint32_t* d_stage2;
  // host (pinned)
  uint2* h_thr; ReplicaObs* h_obs;
  cudaEvent_t thr_copied;
  std::vector<double>* lastT; bool have_T;
  long long launches;
  int sm_count, device;
  bool coop_supported;
  int max_blocks;            // ic_set_max_blocks: 0 = automatic
  int last_family;           // ic_kernel_family: the variant number of the kernels the last sweep call ran (0: none yet)
};
static long long blocks_cap(const ic_ctx* c, long long automatic) {
  return c->max_blocks > 0 ? std::min<long long>(automatic, c->max_blocks) : automatic;
}

static thread_local char g_cuda_msg[256] = "no CUDA error recorded";

static int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "%s: %s", what, cudaGetErrorString(e));
  return IC_ERR_CUDA;
}
#define IC_CUDA(call)                                        \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);      \
  } while (0)

// every entry point that touches the device first makes the context's device current (a caller may have switched)
#define IC_ENTER(c)                                                                \
  do {                                                                             \
    int dev_ = -1;                                                                 \
    if (cudaGetDevice(&dev_) != cudaSuccess || dev_ != (c)->device) IC_CUDA(cudaSetDevice((c)->device)); \
  } while (0)

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
static bool valid_dims(int L, int replicas, int bits) {
  return L >= 4 && L <= 65536 && (L & (L - 1)) == 0 && replicas >= 1 && replicas <= 65535 && (bits == 8 || bits == 2);
}
static size_t lattice_bytes(int L, int bits) { return (size_t)L * L * bits / 8; }

extern "C" size_t ic_workspace_bytes(int L, int replicas, int bits) {
  if (!valid_dims(L, replicas, bits)) return 0;
  size_t b = 0;
  b += align256(lattice_bytes(L, bits)) * (size_t)replicas;       // lattices
  b += align256((size_t)replicas * THR_STRIDE * sizeof(uint2));    // class tables (threshold, packed deltas)
  b += align256(2 * DESC_ENTRIES * sizeof(uint2));                 // move descriptors, FAR and NEAR
  b += align256(2 * ST_DESC_ENTRIES * sizeof(uint2));              // move descriptors of the staged kernels
  b += align256((size_t)replicas * sizeof(ReplicaObs));            // integers and sums
  b += 256;                                                        // scratch for ic_debug_recompute
  b += align256((size_t)replicas * sizeof(CoopScratch));           // per-sweep sums and barrier counters of the one-launch kernel
  b += align256((size_t)replicas * TASK_CTR_STRIDE * 4);           // task counters of the staged kernels
  b += align256((size_t)L * L);                                    // staging of one lattice in public byte codes
  b += align256((size_t)L * L / 4);                                // ... and in packed public codes (ic_set_state_packed / ic_state_packed)
  return b;
}

// U2: acceptance threshold of a class at temperature T.  Metropolis min(1, exp(-dE/T)) as a 29-bit
// integer; IEEE fp64, the C library's exp, no FMA contraction (built with -ffp-contract=off).
static uint32_t threshold29(double delta, double V, double quarterJ, int dn2, int dV, int dJ, double T) {
  const double dE = (delta * (double)dn2 + V * (double)dV) + quarterJ * (double)dJ;
  if (dE <= 0.0) return 1u << 29;
  double t = std::floor(std::exp(-dE / T) * 536870912.0);
  if (t < 1.0) t = 1.0;
  if (t > 536870911.0) t = 536870911.0;
  return (uint32_t)t;
}
static void build_thresholds(const ic_ctx* c, double T, uint32_t* out) {
  const double qJ = 0.25 * c->J;
  for (int a = -1; a <= 1; ++a)
    for (int v = -16; v <= 16; ++v)
      for (int j = -16; j <= 16; ++j) out[class_index_public(2 * a, v, j)] = threshold29(c->delta, c->V, qJ, 2 * a, v, j, T);
}
// Device form of the class table: (8*t29 - 1, packed (dn2, dV, dJ)); w <= 8*t29 - 1  <=>  (w >> 3) < t29.
static void build_class_table(const ic_ctx* c, double T, uint2* out) {
  uint32_t t29[N_CLASSES];
  build_thresholds(c, T, t29);
  for (int k = 0; k < THR_STRIDE; ++k) { out[k].x = 0u; out[k].y = 0u; }
  for (int a = -1; a <= 1; ++a)
    for (int v = -16; v <= 16; ++v)
      for (int j = -16; j <= 16; ++j) {
        const int k = class_index(2 * a, v, j);
        out[k].x = 8u * t29[class_index_public(2 * a, v, j)] - 1u;
        out[k].y = (uint32_t)pack_delta(2 * a, v, j);
      }
}

// The table of two-site configurations in the paper's listing order, as move descriptors for the
// tiled kernels.  Entry [key*8 + r], key = fa | fb<<1 | ga<<3 | gb<<4 in the (f,g) site encoding of LAY_P16:
//   x = int8 x 4 (cFa, cGa, cFb, cGb): class index = K + cFa*Fa + cGa*Ga + cFb*Fb + cGb*Gb, where the neighbour sums are
//       sum S = F+G-4, sum sigma = F-G, i.e. cF = CLS_SB*dS + dsig, cG = CLS_SB*dS - dsig (the -4 cancels: dS_a + dS_b = 0);
//   y = 8*K | (xor of the site bytes: a at bits 0,3, b at bits 1,4) << 16 | (dM & 15 | (dD & 15) << 4) << 24,
//       K = class_index(E_Delta, adj*dS_a*dS_b, adj*dsig_a*dsig_b)  (eq. 4 for adj = 0, eq. 5 for adj = 1),
//       dM = dsig_a + dsig_b, dD = dsig_a - dsig_b.
// Null proposals (q = +-2, r >= 6 for q = 0, the current configuration) have x = 0, no change and the class entry
// NULL_CLASS (threshold 0: never "accepted", see ic_common.cuh).
static void build_descriptors(int adj, uint2* out) {
  static const int Q0[6][2] = {{2, 3}, {3, 2}, {0, 0}, {1, 1}, {0, 1}, {1, 0}};
  for (int key = 0; key < 28; ++key)
    for (int r = 0; r < 8; ++r) {
      uint2 d; d.x = 0u; d.y = 8u * (uint32_t)NULL_CLASS;
      const int ea = (key & 1) | (key & 8), eb = ((key >> 1) & 1) | ((key >> 1) & 8);
      const bool valid = (key & ~0x1B) == 0;
      if (valid) {
        const int ca = code_of_e(ea), cb = code_of_e(eb);
        const int q = S_of(ca) + S_of(cb);
        int na = ca, nb = cb;
        if (q == 0) { if (r < 6) { na = Q0[r][0]; nb = Q0[r][1]; } }
        else if (q == 1 || q == -1) {
          const int C = q > 0 ? 2 : 3;
          switch (r & 3) { case 0: na = C; nb = 0; break; case 1: na = C; nb = 1; break; case 2: na = 0; nb = C; break; default: na = 1; nb = C; }
        }
        if (na != ca || nb != cb) {
          const int dSa = S_of(na) - S_of(ca), dSb = S_of(nb) - S_of(cb), dGa = sg_of(na) - sg_of(ca), dGb = sg_of(nb) - sg_of(cb);
          const int e_d = S_of(na) * S_of(na) + S_of(nb) * S_of(nb) - S_of(ca) * S_of(ca) - S_of(cb) * S_of(cb);
          const int K = class_index(e_d, adj * dSa * dSb, adj * dGa * dGb);
          const int cf[4] = {CLS_SB * dSa + dGa, CLS_SB * dSa - dGa, CLS_SB * dSb + dGb, CLS_SB * dSb - dGb};
          d.x = 0u;
          for (int k = 0; k < 4; ++k) d.x |= ((uint32_t)(cf[k] & 0xFF)) << (8 * k);
          const int xa = ea ^ e_of_code(na), xb = eb ^ e_of_code(nb);
          const int dM = dGa + dGb, dD = dGa - dGb;
          d.y = 8u * (uint32_t)K | ((uint32_t)(xa | (xb << 1)) << 16) | ((uint32_t)((dM & 15) | ((dD & 15) << 4)) << 24);
        }
      }
      out[key * 8 + r] = d;
    }
}

// The same table for the staged kernels, entry [adj][key*8 + r] = (coef, info):
//   coef = the four int8 coefficients (cFa, cGa/2, cFb, cGb/2); info = 4*K (byte offset of the class base in the 4-byte threshold table) |
//   (xor of the site bytes: a at bits 0,3, b at bits 1,4) << 16.
static void build_descriptors32(uint2* out) {
  std::vector<uint2> d8(DESC_ENTRIES);
  for (int adj = 0; adj < 2; ++adj) {
    build_descriptors(adj, d8.data());
    for (int e = 0; e < ST_DESC_ENTRIES; ++e) {
      uint2 q; q.x = 0u; q.y = 4u * (uint32_t)NULL_CLASS;
      if (e < DESC_ENTRIES) {
        const uint2 d = d8[e];
        // the kernel feeds (4F, 8G) per site: halve the G coefficients (CLS_SB dS - dsig is even: CLS_SB is odd)
        const int cFa = (int8_t)(d.x & 0xFF), cGa = (int8_t)((d.x >> 8) & 0xFF), cFb = (int8_t)((d.x >> 16) & 0xFF), cGb = (int8_t)((d.x >> 24) & 0xFF);
        q.x = (uint32_t)(cFa & 0xFF) | ((uint32_t)((cGa / 2) & 0xFF) << 8) | ((uint32_t)(cFb & 0xFF) << 16) | ((uint32_t)((cGb / 2) & 0xFF) << 24);
        q.y = ((d.y & 0xFFFFu) >> 1) | (((d.y >> 16) & 0xFFu) << 16);
      }
      out[adj * ST_DESC_ENTRIES + e] = q;
    }
  }
}

// U4: parameters of sweep s, from Philox(ctr = (0, 0, s, TAG_SCHED), key = seed); the same for all replicas.
static void schedule_params(int L, uint64_t seed, uint64_t sweep, int32_t out4[4]) {
  u32x4 z = philox4x32_10(0u, 0u, (uint32_t)sweep, TAG_SCHED << 28, (uint32_t)seed, (uint32_t)(seed >> 32));
  if ((sweep & 1) == 0) {   // FAR sweep: odd XOR masks, partner(x,y) = (x^mx, y^my)
    out4[0] = 0; out4[1] = (int32_t)(2 * (z.v[0] & (uint32_t)(L / 2 - 1)) + 1); out4[2] = (int32_t)(2 * (z.v[1] & (uint32_t)(L / 2 - 1)) + 1);
  } else {                  // NEAR sweep: dominoes, orientation and offset
    out4[0] = 1; out4[1] = (int32_t)(z.v[0] & 1u); out4[2] = (int32_t)(z.v[1] & 3u);
  }
  out4[3] = 0;
}

// U0, stage 1: all sites magnetic with random sigma, then nplus sites S=+1 and nminus sites S=-1
// at distinct random sites by selection sampling over the counter-based stream (seed, replica, TAG_INIT).
static void stage1_init(int8_t* code, long long N, long long nplus, long long nminus, uint64_t seed, int replica) {
  const long long CH = 1LL << 20;
  unsigned hw = std::thread::hardware_concurrency();
  const int nth = (int)std::max(1u, std::min(hw ? hw : 1u, 32u));
  std::vector<uint32_t> w(3 * (size_t)std::min(CH, N));
  const long long K = nplus + nminus;
  long long picked = 0, plus = 0;
  for (long long base = 0; base < N; base += CH) {
    const long long cnt = std::min(CH, N - base);
    auto fill = [&](long long lo, long long hi) {
      for (long long k = lo; k < hi; ++k) {
        const long long i = base + k;
        u32x4 z = philox4x32_10((uint32_t)(i & 0xFFFFFFFFLL), (uint32_t)(i >> 32), 0u,
                                ((uint32_t)replica & 0x0FFFFFFFu) | (TAG_INIT << 28), (uint32_t)seed, (uint32_t)(seed >> 32));
        w[3 * k] = z.v[0]; w[3 * k + 1] = z.v[1]; w[3 * k + 2] = z.v[2];
      }
    };
    if (cnt < 65536 || nth == 1) fill(0, cnt);
    else {
      std::vector<std::thread> th;
      for (int t = 0; t < nth; ++t) th.emplace_back(fill, cnt * t / nth, cnt * (t + 1) / nth);
      for (auto& t : th) t.join();
    }
    for (long long k = 0; k < cnt; ++k) {
      const long long i = base + k;
      int c = (w[3 * k] & 1u) ? 1 : 0;
      if ((long long)(((uint64_t)w[3 * k + 1] * (uint64_t)(N - i)) >> 32) < K - picked) {
        if ((long long)(((uint64_t)w[3 * k + 2] * (uint64_t)(K - picked)) >> 32) < nplus - plus) { c = 2; ++plus; }
        else c = 3;
        ++picked;
      }
      code[i] = (int8_t)c;
    }
  }
}

__global__ void k_store_ints(ReplicaObs* o, const long long* s8) {
  o->n2 = s8[0]; o->bV = s8[1]; o->bJ = s8[2]; o->M = s8[3]; o->Ms = s8[4]; o->Q = s8[5];
}

static int recompute_into_scratch(ic_ctx* c, int replica) {
  IC_CUDA(cudaMemsetAsync(c->d_scratch8, 0, 64, c->stream));
  const LatView lat{c->lattice + (long long)replica * c->lat_stride, c->L, c->logL};
  const int blocks = (int)std::min<long long>((c->N + 255) / 256, (long long)c->sm_count * 8);
  if (c->layout == LAY_ROW8) k_recompute<LAY_ROW8><<<blocks, 256, 0, c->stream>>>(lat, c->d_scratch8);
  else if (c->layout == LAY_ROW2) k_recompute<LAY_ROW2><<<blocks, 256, 0, c->stream>>>(lat, c->d_scratch8);
  else if (c->layout == LAY_P16) k_recompute_p16<8><<<blocks, 256, 0, c->stream>>>((const uint8_t*)lat.base, c->logL, c->d_scratch8);
  else k_recompute_p16<2><<<blocks, 256, 0, c->stream>>>((const uint8_t*)lat.base, c->logL, c->d_scratch8);
  c->launches++;
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}

// Uploads public byte codes (host) into the replica's lattice and refreshes its exact integers.  With `validate` the
// codes are first checked on the device in the staging buffer (every code in 0..3, sum S == Q: eq. 2); a
// rejected lattice leaves the replica untouched.
static int install_staged_codes(ic_ctx* c, int replica);
static int upload_state(ic_ctx* c, int replica, const int8_t* h_codes, bool validate) {
  char* lat = c->lattice + (long long)replica * c->lat_stride;
  const long long n16 = c->N / 16;
  const int blocks = (int)std::min<long long>((n16 + 255) / 256, (long long)c->sm_count * 16);
  IC_CUDA(cudaMemcpyAsync(c->d_stage, h_codes, (size_t)c->N, cudaMemcpyHostToDevice, c->stream));
  if (validate) {
    IC_CUDA(cudaMemsetAsync(c->d_scratch8, 0, 64, c->stream));
    k_validate_codes<<<blocks, 256, 0, c->stream>>>(c->d_stage, n16, c->d_scratch8);
    c->launches++;
    IC_CUDA(cudaGetLastError());
    long long h[2];
    IC_CUDA(cudaMemcpyAsync(h, c->d_scratch8, 16, cudaMemcpyDeviceToHost, c->stream));
    IC_CUDA(cudaStreamSynchronize(c->stream));
    if (h[0] != 0 || h[1] != c->Q) return IC_ERR_CHARGE;
  }
  return install_staged_codes(c, replica);
}
// the lattice in public byte codes in the staging buffer -> the replica's layout; recomputes its exact integers
static int install_staged_codes(ic_ctx* c, int replica) {
  char* lat = c->lattice + (long long)replica * c->lat_stride;
  const long long n16 = c->N / 16;
  const int blocks = (int)std::min<long long>((n16 + 255) / 256, (long long)c->sm_count * 16);
  if (c->layout == LAY_ROW8) IC_CUDA(cudaMemcpyAsync(lat, c->d_stage, (size_t)c->N, cudaMemcpyDeviceToDevice, c->stream));
  else {
    if (c->layout == LAY_ROW2) k_pack2<<<blocks, 256, 0, c->stream>>>(c->d_stage, (uint32_t*)lat, n16);
    else if (c->layout == LAY_P2) k_codes_to_p2<<<std::max(1, blocks / 4), 256, 0, c->stream>>>(c->d_stage, (uint8_t*)lat, c->logL);
    else k_codes_to_p16<<<blocks, 256, 0, c->stream>>>(c->d_stage, (uint8_t*)lat, c->logL);
    c->launches++;
    IC_CUDA(cudaGetLastError());
  }
  int rc = recompute_into_scratch(c, replica);
  if (rc != IC_OK) return rc;
  k_store_ints<<<1, 1, 0, c->stream>>>(&c->d_obs[replica], c->d_scratch8);
  c->launches++;
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}

extern "C" int ic_create(ic_ctx** out, int L, double n, double delta, double V, double J, uint64_t seed, int replicas,
                         int bits, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return IC_ERR_NULL;
  *out = nullptr;
  if (!valid_dims(L, replicas, bits)) return IC_ERR_SIZE;
  if (!std::isfinite(n) || !std::isfinite(delta) || !std::isfinite(V) || !std::isfinite(J) || std::fabs(n) > 1.0) return IC_ERR_PARAM;
  const size_t need = ic_workspace_bytes(L, replicas, bits);
  if (!d_workspace || workspace_bytes < need || ((uintptr_t)d_workspace & 255) != 0) return IC_ERR_WORKSPACE;

  ic_ctx* c = new (std::nothrow) ic_ctx();
  if (!c) return IC_ERR_NULL;
  c->L = L; c->logL = 0; while ((1 << c->logL) < L) c->logL++;
  c->replicas = replicas; c->bits = bits; c->variant = 0; c->max_blocks = 0; c->last_family = 0;
  c->layout = bits == 2 ? (L >= 128 ? LAY_P2 : LAY_ROW2) : (L >= 64 ? LAY_P16 : LAY_ROW8);
  c->N = (long long)L * L; c->Q = std::llround(n * (double)c->N);
  c->n = n; c->delta = delta; c->V = V; c->J = J; c->seed = seed; c->sweep = 0;
  c->stream = (cudaStream_t)cuda_stream;
  c->launches = 0; c->have_T = false; c->lastT = new std::vector<double>((size_t)replicas, 0.0);
  char* p = (char*)d_workspace;
  c->lattice = p; c->lat_stride = (long long)align256(lattice_bytes(L, bits)); p += (size_t)c->lat_stride * replicas;
  c->d_thr = (uint2*)p; p += align256((size_t)replicas * THR_STRIDE * sizeof(uint2));
  c->d_desc = (uint2*)p; p += align256(2 * DESC_ENTRIES * sizeof(uint2));
  c->d_desc32 = (uint2*)p; p += align256(2 * ST_DESC_ENTRIES * sizeof(uint2));
  c->d_obs = (ReplicaObs*)p; p += align256((size_t)replicas * sizeof(ReplicaObs));
  c->d_scratch8 = (long long*)p; p += 256;
  c->d_coop = (CoopScratch*)p; p += align256((size_t)replicas * sizeof(CoopScratch));
  c->d_task_ctr = (unsigned int*)p; p += align256((size_t)replicas * TASK_CTR_STRIDE * 4);
  c->d_stage = (int8_t*)p; p += align256((size_t)c->N);
  c->d_stage2 = (uint32_t*)p;
  c->h_thr = nullptr; c->h_obs = nullptr; c->thr_copied = nullptr;

  auto fail = [&](int rc) { ic_destroy(c); return rc; };
  if (cudaMallocHost((void**)&c->h_thr, (size_t)replicas * THR_STRIDE * sizeof(uint2)) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "cudaMallocHost(thresholds)"));
  if (cudaMallocHost((void**)&c->h_obs, (size_t)replicas * sizeof(ReplicaObs)) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "cudaMallocHost(observables)"));
  if (cudaEventCreateWithFlags(&c->thr_copied, cudaEventDisableTiming) != cudaSuccess) return fail(cuda_fail(cudaGetLastError(), "cudaEventCreate"));
  memset(c->h_thr, 0, (size_t)replicas * THR_STRIDE * sizeof(uint2));
  cudaError_t e = cudaMemsetAsync(c->d_obs, 0, (size_t)replicas * sizeof(ReplicaObs), c->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->d_task_ctr, 0, (size_t)replicas * TASK_CTR_STRIDE * 4, c->stream);
  if (e != cudaSuccess) return fail(cuda_fail(e, "cudaMemsetAsync(observables)"));
  {
    std::vector<uint2> desc(2 * DESC_ENTRIES);
    build_descriptors(0, desc.data()); build_descriptors(1, desc.data() + DESC_ENTRIES);
    e = cudaMemcpyAsync(c->d_desc, desc.data(), desc.size() * sizeof(uint2), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return fail(cuda_fail(e, "upload of the move descriptors"));
    std::vector<uint2> desc32(2 * ST_DESC_ENTRIES);
    build_descriptors32(desc32.data());
    e = cudaMemcpyAsync(c->d_desc32, desc32.data(), desc32.size() * sizeof(uint2), cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return fail(cuda_fail(e, "upload of the staged kernels' move descriptors"));
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
      return fail(cuda_fail(cudaGetLastError(), "cudaDeviceGetAttribute(multiProcessorCount)"));
    c->sm_count = sms; c->device = dev;
    int coop = 0;
    c->coop_supported = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop != 0;
  }

  // stage 1 for every replica
  std::vector<int8_t> codes((size_t)c->N);
  const long long nplus = c->Q > 0 ? c->Q : 0, nminus = c->Q < 0 ? -c->Q : 0;
  for (int r = 0; r < replicas; ++r) {
    stage1_init(codes.data(), c->N, nplus, nminus, seed, r);
    int rc = upload_state(c, r, codes.data(), false);
    if (rc != IC_OK) return fail(rc);
    e = cudaStreamSynchronize(c->stream);   // codes is reused for the next replica
    if (e != cudaSuccess) return fail(cuda_fail(e, "cudaStreamSynchronize(init)"));
  }
  *out = c;
  return IC_OK;
}

extern "C" int ic_destroy(ic_ctx* c) {
  if (!c) return IC_ERR_NULL;
  cudaStreamSynchronize(c->stream);
  if (c->h_thr) cudaFreeHost(c->h_thr);
  if (c->h_obs) cudaFreeHost(c->h_obs);
  if (c->thr_copied) cudaEventDestroy(c->thr_copied);
  delete c->lastT;
  delete c;
  return IC_OK;
}

extern "C" int ic_init_charges(ic_ctx* c, int replica, int64_t nplus, int64_t nminus) {
  if (!c) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  if (nplus < 0 || nminus < 0 || nplus + nminus > c->N || nplus - nminus != c->Q) return IC_ERR_CHARGE;
  IC_ENTER(c);
  std::vector<int8_t> codes((size_t)c->N);
  stage1_init(codes.data(), c->N, nplus, nminus, c->seed, replica);
  int rc = upload_state(c, replica, codes.data(), false);
  if (rc != IC_OK) return rc;
  IC_CUDA(cudaStreamSynchronize(c->stream));
  return IC_OK;
}

extern "C" int ic_set_state(ic_ctx* c, int replica, const int8_t* h_codes) {
  if (!c || !h_codes) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  IC_ENTER(c);
  int rc = upload_state(c, replica, h_codes, true);
  if (rc != IC_OK) return rc;
  IC_CUDA(cudaStreamSynchronize(c->stream));   // h_codes may be pageable and is the caller's to reuse
  return IC_OK;
}

extern "C" int ic_state(ic_ctx* c, int replica, int8_t* h_out) {
  if (!c || !h_out) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  IC_ENTER(c);
  const char* lat = c->lattice + (long long)replica * c->lat_stride;
  if (c->layout == LAY_ROW8) {
    IC_CUDA(cudaMemcpyAsync(h_out, lat, (size_t)c->N, cudaMemcpyDeviceToHost, c->stream));
  } else {
    const long long n16 = c->N / 16;
    const int blocks = (int)std::min<long long>((n16 + 255) / 256, (long long)c->sm_count * 16);
    if (c->layout == LAY_ROW2) k_unpack2<<<blocks, 256, 0, c->stream>>>((const uint32_t*)lat, c->d_stage, n16);
    else if (c->layout == LAY_P2) k_p2_to_codes<<<std::max(1, blocks / 4), 256, 0, c->stream>>>((const uint8_t*)lat, c->d_stage, c->logL);
    else k_p16_to_codes<<<blocks, 256, 0, c->stream>>>((const uint8_t*)lat, c->d_stage, c->logL);
    c->launches++;
    IC_CUDA(cudaGetLastError());
    IC_CUDA(cudaMemcpyAsync(h_out, c->d_stage, (size_t)c->N, cudaMemcpyDeviceToHost, c->stream));
  }
  IC_CUDA(cudaStreamSynchronize(c->stream));
  return IC_OK;
}

// ---- lattices at 2 bits per site over PCIe (a site has four states) -----------------------------------------
// The packed public format is layout ROW2: word i holds the sites 16 i .. 16 i + 15 of the row-major lattice, site k of the
// word in bits 2k, 2k+1.  A quarter of the bytes of ic_set_state / ic_state cross the bus; the conversions run on the device.
extern "C" int ic_set_state_packed(ic_ctx* c, int replica, const uint32_t* h_words) {
  if (!c || !h_words) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  IC_ENTER(c);
  const long long n16 = c->N / 16;
  const int blocks = (int)std::min<long long>((n16 + 255) / 256, (long long)c->sm_count * 16);
  IC_CUDA(cudaMemcpyAsync(c->d_stage2, h_words, (size_t)c->N / 4, cudaMemcpyHostToDevice, c->stream));
  IC_CUDA(cudaMemsetAsync(c->d_scratch8, 0, 64, c->stream));
  k_charge_of_packed<<<blocks, 256, 0, c->stream>>>(c->d_stage2, n16, c->d_scratch8);
  c->launches++;
  IC_CUDA(cudaGetLastError());
  long long h[2];
  IC_CUDA(cudaMemcpyAsync(h, c->d_scratch8, 16, cudaMemcpyDeviceToHost, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  if (h[1] != c->Q) return IC_ERR_CHARGE;                              // the replica is untouched
  if (c->layout == LAY_ROW2) {                                         // the packed format is the layout
    IC_CUDA(cudaMemcpyAsync(c->lattice + (long long)replica * c->lat_stride, c->d_stage2, (size_t)c->N / 4, cudaMemcpyDeviceToDevice, c->stream));
    int rc = recompute_into_scratch(c, replica);
    if (rc != IC_OK) return rc;
    k_store_ints<<<1, 1, 0, c->stream>>>(&c->d_obs[replica], c->d_scratch8);
    c->launches++;
    IC_CUDA(cudaGetLastError());
  } else {
    k_unpack2<<<blocks, 256, 0, c->stream>>>(c->d_stage2, c->d_stage, n16);
    c->launches++;
    IC_CUDA(cudaGetLastError());
    int rc = install_staged_codes(c, replica);
    if (rc != IC_OK) return rc;
  }
  IC_CUDA(cudaStreamSynchronize(c->stream));
  return IC_OK;
}

extern "C" int ic_state_packed(ic_ctx* c, int replica, uint32_t* h_out) {
  if (!c || !h_out) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  IC_ENTER(c);
  const char* lat = c->lattice + (long long)replica * c->lat_stride;
  const long long n16 = c->N / 16;
  const int blocks = (int)std::min<long long>((n16 + 255) / 256, (long long)c->sm_count * 16);
  const void* src = c->d_stage2;
  if (c->layout == LAY_ROW2) src = lat;
  else {
    const int8_t* codes = c->d_stage;
    if (c->layout == LAY_ROW8) codes = (const int8_t*)lat;
    else if (c->layout == LAY_P2) k_p2_to_codes<<<std::max(1, blocks / 4), 256, 0, c->stream>>>((const uint8_t*)lat, c->d_stage, c->logL);
    else k_p16_to_codes<<<blocks, 256, 0, c->stream>>>((const uint8_t*)lat, c->d_stage, c->logL);
    k_pack2<<<blocks, 256, 0, c->stream>>>(codes, c->d_stage2, n16);
    c->launches += c->layout == LAY_ROW8 ? 1 : 2;
    IC_CUDA(cudaGetLastError());
  }
  IC_CUDA(cudaMemcpyAsync(h_out, src, (size_t)c->N / 4, cudaMemcpyDeviceToHost, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  return IC_OK;
}

// Launch as a programmatic dependent of the previous kernel of the stream: the kernel may start while that one drains
// (every phase kernel and the fold call griddepcontrol.wait before they touch anything a kernel writes).
template <class... KArgs, class... Args>
static cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, args...);
}

static int launch_phase_ref(ic_ctx* c, const PhaseArgs& a) {
  const long long npairs = c->N / 4;
  dim3 grid((unsigned)((npairs + 255) / 256), (unsigned)c->replicas);
  if (c->layout == LAY_ROW8) IC_CUDA(launch_pdl(k_ref_phase<LAY_ROW8>, grid, dim3(256), 0, c->stream, a));
  else if (c->layout == LAY_ROW2) IC_CUDA(launch_pdl(k_ref_phase<LAY_ROW2>, grid, dim3(256), 0, c->stream, a));
  else if (c->layout == LAY_P2) IC_CUDA(launch_pdl(k_ref_phase<LAY_P2>, grid, dim3(256), 0, c->stream, a));
  else IC_CUDA(launch_pdl(k_ref_phase<LAY_P16>, grid, dim3(256), 0, c->stream, a));
  c->launches++;
  return IC_OK;
}

// Tiled kernels on LAY_P16: one item (32 pair updates) per thread, persistent blocks over the items of a replica.
static int launch_phase_p16(ic_ctx* c, PhaseArgs a) {
  const long long n_items = c->N / 128;
  const long long nb = (n_items + P16_THREADS - 1) / P16_THREADS;
  const long long cap = blocks_cap(c, std::max<long long>(1, ((long long)c->sm_count * 6 + c->replicas - 1) / c->replicas));
  dim3 grid((unsigned)std::min(nb, cap), (unsigned)c->replicas);
  if (a.type == 0) {
    a.desc = c->d_desc;
    switch (((a.p1 >> 2) & 15) >> 2) {
      case 0: IC_CUDA(launch_pdl(k_p16_phase<PH_FAR, 0>, grid, dim3(P16_THREADS), 0, c->stream, a)); break;
      case 1: IC_CUDA(launch_pdl(k_p16_phase<PH_FAR, 1>, grid, dim3(P16_THREADS), 0, c->stream, a)); break;
      case 2: IC_CUDA(launch_pdl(k_p16_phase<PH_FAR, 2>, grid, dim3(P16_THREADS), 0, c->stream, a)); break;
      default: IC_CUDA(launch_pdl(k_p16_phase<PH_FAR, 3>, grid, dim3(P16_THREADS), 0, c->stream, a)); break;
    }
  } else {
    a.desc = c->d_desc + DESC_ENTRIES;
    if (a.p1 == 0) IC_CUDA(launch_pdl(k_p16_phase<PH_NEAR_H, 0>, grid, dim3(P16_THREADS), 0, c->stream, a));
    else IC_CUDA(launch_pdl(k_p16_phase<PH_NEAR_V, 0>, grid, dim3(P16_THREADS), 0, c->stream, a));
  }
  c->launches++;
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}

// Staged kernels on LAY_P16, L >= 2048: one persistent block per SM, TMA-staged regions (ic_kernels_staged.cuh).
template <int TYPE, int CW, int BITS>
static int launch_staged_bits(ic_ctx* c, const PhaseArgs& a, dim3 grid) {
  using C = StagedCfg<TYPE, BITS>;
  static std::atomic<bool> configured[64] = {};   // per instantiation and per device: the attribute belongs to the device's copy of the kernel
  if (c->device < 0 || c->device >= 64 || !configured[c->device]) {
    IC_CUDA(cudaFuncSetAttribute(k_staged_phase<TYPE, CW, BITS>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    if (c->device >= 0 && c->device < 64) configured[c->device] = true;
  }
  IC_CUDA(launch_pdl(k_staged_phase<TYPE, CW, BITS>, grid, dim3(ST_THREADS), (size_t)C::SMEM_BYTES, c->stream, a));
  return IC_OK;
}
template <int TYPE, int CW>
static int launch_staged_one(ic_ctx* c, const PhaseArgs& a, dim3 grid) {
  return c->layout == LAY_P2 ? launch_staged_bits<TYPE, CW, 2>(c, a, grid) : launch_staged_bits<TYPE, CW, 8>(c, a, grid);
}
// one cooperative launch for all the sweeps of a call: single mid-size lattices (ic_kernels_coop.cuh)
static bool coop_ok(const ic_ctx* c) {
  return (c->layout == LAY_P16 || c->layout == LAY_P2) && c->L >= COOP_MIN_L && c->L <= COOP_MAX_L && c->coop_supported;
}
template <int BITS>
static int launch_coop(ic_ctx* c, int64_t nsweeps, int64_t* d_trace) {
  static std::atomic<bool> configured[64] = {};
  if (c->device < 0 || c->device >= 64 || !configured[c->device]) {
    IC_CUDA(cudaFuncSetAttribute(k_coop_sweeps<BITS>, cudaFuncAttributeMaxDynamicSharedMemorySize, COOP_SMEM_BYTES));
    if (c->device >= 0 && c->device < 64) configured[c->device] = true;
  }
  CoopArgs a;
  a.lattice = c->lattice; a.thr = c->d_thr; a.desc32 = c->d_desc32; a.obs = c->d_obs; a.scratch = c->d_coop; a.trace = (long long*)d_trace;
  a.lat_stride = c->lat_stride; a.nsweeps = nsweeps; a.sweep0 = c->sweep; a.delta = c->delta; a.V = c->V; a.quarterJ = 0.25 * c->J;
  a.L = c->L; a.logL = c->logL; a.replicas = c->replicas; a.key0 = (uint32_t)c->seed; a.key1 = (uint32_t)(c->seed >> 32);
  const long long items = c->N / 16;                                   // four pairs per item, N/4 pairs per phase
  // latency-bound: spread the items of a phase over as many SMs as there are, at least four warps per block
  const int rows = std::min(c->replicas, c->sm_count);              // rows of blocks; a row takes every rows-th replica
  const long long cap = blocks_cap(c, std::max<long long>(1, c->sm_count / rows));
  const long long nblk = std::min(cap, (items + 127) / 128);
  // item threads per block + the service warp
  const int threads = 32 + (int)std::min<long long>(COOP_THREADS - 32, std::max<long long>(128, ((items + nblk - 1) / nblk + 31) / 32 * 32));
  dim3 grid((unsigned)nblk, (unsigned)rows);
  IC_CUDA(cudaMemsetAsync(c->d_coop, 0, (size_t)c->replicas * sizeof(CoopScratch), c->stream));
  static_assert(COOP_BAR_BASE == 0xFFFFFFFFu, "the barrier counters are set bytewise");
  IC_CUDA(cudaMemset2DAsync(&c->d_coop->arrived, sizeof(CoopScratch), 0xFF, sizeof(unsigned int), (size_t)c->replicas, c->stream));
  void* args[] = {(void*)&a};
  cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_coop_sweeps<BITS>, grid, dim3(threads), args, (size_t)COOP_SMEM_BYTES, c->stream);
  // fewer SMs available than the device reports (MPS, green contexts): the results do not depend on the number of blocks
  // per replica, so try again with half as many before giving the kernel up
  while (e == cudaErrorCooperativeLaunchTooLarge && grid.x > 1) {
    (void)cudaGetLastError();
    grid.x = (grid.x + 1) / 2;
    e = cudaLaunchCooperativeKernel((const void*)k_coop_sweeps<BITS>, grid, dim3(threads), args, (size_t)COOP_SMEM_BYTES, c->stream);
  }
  if (e == cudaErrorCooperativeLaunchTooLarge) {   // not even one block per row of replicas fits
    (void)cudaGetLastError();
    if (c->variant == 5) return cuda_fail(e, "ic_set_variant(5) was asked for, but the one-launch kernel does not fit this GPU partition");
    c->coop_supported = false;                     // automatic selection: the per-phase kernels from now on
    return 1;
  }
  IC_CUDA(e);
  c->launches++;
  return IC_OK;
}
// small lattices: one block per replica, lattice resident in shared memory, the items of the one-launch kernel
static bool resvec_ok(const ic_ctx* c) { return c->L >= RESV_MIN_L && c->L <= RESV_MAX_L; }
template <int LAYG>
static int launch_resvec(ic_ctx* c, int64_t nsweeps, int64_t* d_trace) {
  static std::atomic<bool> configured[64] = {};
  if (c->device < 0 || c->device >= 64 || !configured[c->device]) {
    IC_CUDA(cudaFuncSetAttribute(k_resvec_sweeps<LAYG>, cudaFuncAttributeMaxDynamicSharedMemorySize, RESV_SMEM_BYTES));
    if (c->device >= 0 && c->device < 64) configured[c->device] = true;
  }
  CoopArgs a;
  a.lattice = c->lattice; a.thr = c->d_thr; a.desc32 = c->d_desc32; a.obs = c->d_obs; a.scratch = c->d_coop; a.trace = (long long*)d_trace;
  a.lat_stride = c->lat_stride; a.nsweeps = nsweeps; a.sweep0 = c->sweep; a.delta = c->delta; a.V = c->V; a.quarterJ = 0.25 * c->J;
  a.L = c->L; a.logL = c->logL; a.replicas = c->replicas; a.key0 = (uint32_t)c->seed; a.key1 = (uint32_t)(c->seed >> 32);
  const long long items = c->N / 16;
  const int threads = 32 + (int)std::min<long long>(COOP_THREADS - 32, std::max<long long>(32, (items + 31) / 32 * 32));   // + the service warp
  k_resvec_sweeps<LAYG><<<c->replicas, threads, RESV_SMEM_BYTES, c->stream>>>(a);
  c->launches++;
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}
static bool staged_ok(const ic_ctx* c) { return (c->layout == LAY_P16 || c->layout == LAY_P2) && c->L >= 4 * ST_SEG; }
static bool tiled_ok(const ic_ctx* c) { return c->layout == LAY_P16 && c->L <= 4 * ST_SEG; }   // one tile per row quad
static int launch_phase_staged(ic_ctx* c, PhaseArgs a) {
  const long long ntasks = ((long long)(c->L / 4) * (c->L / 4 / ST_SEG)) / 2;
  const long long cap = blocks_cap(c, std::max<long long>(1, c->sm_count / c->replicas));
  dim3 grid((unsigned)std::min(ntasks, cap), (unsigned)c->replicas);
  a.desc32 = c->d_desc32;
  // Philox: the ten round keys and the parts of the first two rounds that are the same for the whole launch (U3)
  for (int i = 0; i < 10; ++i) { a.rk[2 * i] = a.key0 + (uint32_t)i * PHILOX_W0; a.rk[2 * i + 1] = a.key1 + (uint32_t)i * PHILOX_W1; }
  {
    uint32_t h, l;
    mulhilo(PHILOX_M1, a.c2, h, l);
    a.f0 = h ^ a.rk[0]; a.f1 = l; a.f2 = l ^ a.rk[2];
  }
  int rc;
  if (a.type == 0) {
    switch (((a.p1 >> 2) & 15) >> 2) {
      case 0: rc = launch_staged_one<PH_FAR, 0>(c, a, grid); break;
      case 1: rc = launch_staged_one<PH_FAR, 1>(c, a, grid); break;
      case 2: rc = launch_staged_one<PH_FAR, 2>(c, a, grid); break;
      default: rc = launch_staged_one<PH_FAR, 3>(c, a, grid); break;
    }
  } else if (a.p1 == 0) rc = launch_staged_one<PH_NEAR_H, 0>(c, a, grid);
  else rc = launch_staged_one<PH_NEAR_V, 0>(c, a, grid);
  if (rc != IC_OK) return rc;
  c->launches++;
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}

// thresholds: rebuilt and uploaded only when a temperature changed
static int ensure_thresholds(ic_ctx* c, const double* h_T) {
  bool changed = !c->have_T;
  for (int r = 0; r < c->replicas && !changed; ++r) changed = (*c->lastT)[r] != h_T[r];
  if (changed) {
    IC_CUDA(cudaEventSynchronize(c->thr_copied));   // the previous upload has left the pinned buffer
    for (int r = 0; r < c->replicas; ++r) {
      if (c->have_T && (*c->lastT)[r] == h_T[r]) continue;
      build_class_table(c, h_T[r], c->h_thr + (size_t)r * THR_STRIDE);
      (*c->lastT)[r] = h_T[r];
    }
    IC_CUDA(cudaMemcpyAsync(c->d_thr, c->h_thr, (size_t)c->replicas * THR_STRIDE * sizeof(uint2), cudaMemcpyHostToDevice, c->stream));
    IC_CUDA(cudaEventRecord(c->thr_copied, c->stream));
    c->have_T = true;
  }

  return IC_OK;
}

static int sweep_impl(ic_ctx* c, const double* h_T, int64_t nsweeps, int64_t* d_trace) {
  if (!c || !h_T) return IC_ERR_NULL;
  if (nsweeps < 0 || c->sweep + (uint64_t)nsweeps >= (1ull << 31)) return IC_ERR_PARAM;
  for (int r = 0; r < c->replicas; ++r)
    if (!(h_T[r] > 0.0) || !std::isfinite(h_T[r])) return IC_ERR_PARAM;
  if (nsweeps == 0) return IC_OK;

  IC_ENTER(c);
  { int rc = ensure_thresholds(c, h_T); if (rc != IC_OK) return rc; }

  // small lattices: all the sweeps in one launch, one block per replica, lattice resident in shared memory
  if (resvec_ok(c) && (c->variant == 0 || c->variant == 6)) {
    int rc = c->layout == LAY_ROW8 ? launch_resvec<LAY_ROW8>(c, nsweeps, d_trace)
             : c->layout == LAY_ROW2 ? launch_resvec<LAY_ROW2>(c, nsweeps, d_trace) : launch_resvec<LAY_P16>(c, nsweeps, d_trace);
    if (rc != IC_OK) return rc;
    c->sweep += (uint64_t)nsweeps; c->last_family = 6;
    return IC_OK;
  }
  if (c->L <= RES_MAX_L && (c->variant == 0 || c->variant == 4)) {
    ResidentArgs ra;
    ra.lattice = c->lattice; ra.thr = c->d_thr; ra.obs = c->d_obs; ra.trace = (long long*)d_trace; ra.lat_stride = c->lat_stride;
    ra.nsweeps = nsweeps; ra.sweep0 = c->sweep; ra.delta = c->delta; ra.V = c->V; ra.quarterJ = 0.25 * c->J;
    ra.L = c->L; ra.logL = c->logL; ra.replicas = c->replicas; ra.key0 = (uint32_t)c->seed; ra.key1 = (uint32_t)(c->seed >> 32);
    const int rthreads = (int)std::min<long long>(RES_THREADS, std::max<long long>(64, (c->N / 4 + 31) / 32 * 32));   // one per pair of a phase
    if (c->layout == LAY_ROW8) k_resident_sweeps<LAY_ROW8><<<c->replicas, rthreads, 0, c->stream>>>(ra);
    else if (c->layout == LAY_ROW2) k_resident_sweeps<LAY_ROW2><<<c->replicas, rthreads, 0, c->stream>>>(ra);
    else k_resident_sweeps<LAY_P16><<<c->replicas, rthreads, 0, c->stream>>>(ra);
    c->launches++;
    IC_CUDA(cudaGetLastError());
    c->sweep += (uint64_t)nsweeps; c->last_family = 4;
    return IC_OK;
  }

  // single mid-size lattices: all the sweeps in one cooperative launch over the whole GPU
  if (coop_ok(c) && (c->variant == 0 || c->variant == 5)) {
    int rc = c->layout == LAY_P2 ? launch_coop<2>(c, nsweeps, d_trace) : launch_coop<8>(c, nsweeps, d_trace);
    if (rc < 0) return rc;
    if (rc == IC_OK) { c->sweep += (uint64_t)nsweeps; c->last_family = 5; return IC_OK; }
    // rc > 0 (automatic selection only): the cooperative launch does not fit; fall through to the phase kernels
  }

  PhaseArgs a;
  a.lattice = c->lattice; a.thr = c->d_thr; a.desc = c->d_desc; a.desc32 = c->d_desc32; a.obs = c->d_obs; a.lat_stride = c->lat_stride;
  a.L = c->L; a.logL = c->logL; a.key0 = (uint32_t)c->seed; a.key1 = (uint32_t)(c->seed >> 32);
  const double qJ = 0.25 * c->J;
  for (int64_t s = 0; s < nsweeps; ++s) {
    int32_t par[4];
    schedule_params(c->L, c->seed, c->sweep, par);
    a.type = par[0]; a.p1 = par[1]; a.p2 = par[2];
    bool absolute = false;
    for (int phase = 0; phase < 2; ++phase) {
      a.phase = phase; a.c2 = (uint32_t)(2 * c->sweep + (uint64_t)phase); a.task_ctr = c->d_task_ctr + phase;
      const bool staged = staged_ok(c) && (c->variant == 3 || c->variant == 0);
      const bool tiled = tiled_ok(c) && (c->variant == 0 || c->variant == 2);
      absolute = staged;     // the staged kernels report M, Ms of the updated sites instead of their changes
      c->last_family = staged ? 3 : tiled ? 2 : 1;
      int rc = staged ? launch_phase_staged(c, a) : tiled ? launch_phase_p16(c, a) : launch_phase_ref(c, a);
      if (rc != IC_OK) return rc;
    }
    {
      long long* trow = d_trace ? (long long*)d_trace + 6LL * c->replicas * s : nullptr;
      IC_CUDA(launch_pdl(k_fold, dim3((unsigned)((c->replicas + 127) / 128)), dim3(128), 0, c->stream, c->d_obs, c->replicas, c->delta, c->V, qJ, trow, absolute ? 1 : 0, c->d_task_ctr));
    }
    c->launches++;
    IC_CUDA(cudaGetLastError());
    c->sweep += 1;
  }
  return IC_OK;
}

extern "C" int ic_sweep(ic_ctx* c, const double* h_T, int64_t nsweeps) { return sweep_impl(c, h_T, nsweeps, nullptr); }
extern "C" int ic_sweep_trace(ic_ctx* c, const double* h_T, int64_t nsweeps, int64_t* d_trace) {
  if (!d_trace && nsweeps > 0) return IC_ERR_NULL;
  return sweep_impl(c, h_T, nsweeps, d_trace);
}

__global__ void k_reset_sums(ReplicaObs* obs, int replicas) {
  int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= replicas) return;
  ReplicaObs* o = &obs[r];
  o->nmeas = 0; o->sumE = o->sumE2 = o->sumM = o->sumM2 = o->sumAbsM = o->sumMs = o->sumMs2 = o->sumAbsMs = 0.0;
}

extern "C" int ic_reset_observables(ic_ctx* c) {
  if (!c) return IC_ERR_NULL;
  IC_ENTER(c);
  k_reset_sums<<<(c->replicas + 127) / 128, 128, 0, c->stream>>>(c->d_obs, c->replicas);
  c->launches++;
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}

extern "C" int ic_observables(ic_ctx* c, ic_obs* h_out) {
  if (!c || !h_out) return IC_ERR_NULL;
  IC_ENTER(c);
  IC_CUDA(cudaMemcpyAsync(c->h_obs, c->d_obs, (size_t)c->replicas * sizeof(ReplicaObs), cudaMemcpyDeviceToHost, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  for (int r = 0; r < c->replicas; ++r) {
    const ReplicaObs& o = c->h_obs[r];
    ic_obs& q = h_out[r];
    q.nmeas = o.nmeas; q.n2 = o.n2; q.bV = o.bV; q.bJ = o.bJ; q.M = o.M; q.Ms = o.Ms; q.Q = o.Q;
    q.sumE = o.sumE; q.sumE2 = o.sumE2; q.sumM = o.sumM; q.sumM2 = o.sumM2; q.sumAbsM = o.sumAbsM;
    q.sumMs = o.sumMs; q.sumMs2 = o.sumMs2; q.sumAbsMs = o.sumAbsMs;
    const double T = c->have_T ? (*c->lastT)[r] : 0.0;
    q.T = T; q.C = q.chi_u = q.chi_s = 0.0;
    if (T > 0.0) {   // C = (<E^2> - <E>^2)/(N k T^2), k = 1; chi: DESIGN.md G9
      const double cnt = (double)(o.nmeas > 0 ? o.nmeas : 1), Nd = (double)c->N;
      const double mE = o.sumE / cnt, mE2 = o.sumE2 / cnt, mM = o.sumM / cnt, mM2 = o.sumM2 / cnt;
      const double mMs = o.sumMs / cnt, mMs2 = o.sumMs2 / cnt;
      q.C = (mE2 - mE * mE) / (Nd * T * T);
      q.chi_u = (mM2 - mM * mM) / (Nd * T);
      q.chi_s = (mMs2 - mMs * mMs) / (Nd * T);
    }
  }
  return IC_OK;
}

// Resume (lattice + global sweep counter + seed determine the future; the fp64 sums continue the averages).
extern "C" int ic_restore(ic_ctx* c, int64_t sweep_count, const ic_obs* h_in) {
  if (!c || !h_in) return IC_ERR_NULL;
  if (sweep_count < 0 || (uint64_t)sweep_count >= (1ull << 31)) return IC_ERR_PARAM;
  for (int r = 0; r < c->replicas; ++r) {
    const ic_obs& q = h_in[r];
    const double v[8] = {q.sumE, q.sumE2, q.sumM, q.sumM2, q.sumAbsM, q.sumMs, q.sumMs2, q.sumAbsMs};
    if (q.nmeas < 0) return IC_ERR_PARAM;
    for (double x : v) if (!std::isfinite(x)) return IC_ERR_PARAM;
  }
  IC_ENTER(c);
  // the integers of the current lattices stay as they are (ic_set_state recomputed them); only nmeas and the sums change
  IC_CUDA(cudaMemcpyAsync(c->h_obs, c->d_obs, (size_t)c->replicas * sizeof(ReplicaObs), cudaMemcpyDeviceToHost, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  for (int r = 0; r < c->replicas; ++r) {
    ReplicaObs& o = c->h_obs[r];
    const ic_obs& q = h_in[r];
    o.nmeas = q.nmeas; o.sumE = q.sumE; o.sumE2 = q.sumE2; o.sumM = q.sumM; o.sumM2 = q.sumM2; o.sumAbsM = q.sumAbsM;
    o.sumMs = q.sumMs; o.sumMs2 = q.sumMs2; o.sumAbsMs = q.sumAbsMs;
  }
  IC_CUDA(cudaMemcpyAsync(c->d_obs, c->h_obs, (size_t)c->replicas * sizeof(ReplicaObs), cudaMemcpyHostToDevice, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  c->sweep = (uint64_t)sweep_count;
  return IC_OK;
}

extern "C" int ic_debug_recompute(ic_ctx* c, int replica, int64_t* out6) {
  if (!c || !out6) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  IC_ENTER(c);
  int rc = recompute_into_scratch(c, replica);
  if (rc != IC_OK) return rc;
  long long h[8];
  IC_CUDA(cudaMemcpyAsync(h, c->d_scratch8, 64, cudaMemcpyDeviceToHost, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  for (int k = 0; k < 6; ++k) out6[k] = h[k];
  return IC_OK;
}


// ---- maps -----------------------------------------------------------------------------------------
static bool small_index_ok(const ic_ctx* c) { return c->L <= 32768; }   // site indices as int32

extern "C" size_t ic_maps_scratch_bytes(int L, int64_t K) {
  if (L < 4 || L > 32768 || (L & (L - 1)) || K < 1 || K > (1LL << 30)) return 0;
  return align256((size_t)L * L * 4) + align256((size_t)K * 8) + 256;
}

extern "C" int ic_sweep_maps(ic_ctx* c, const double* h_T, int64_t nmaps, int64_t K, void* d_scratch, size_t scratch_bytes,
                             int64_t* d_trace) {
  if (!c || !h_T) return IC_ERR_NULL;
  if (!small_index_ok(c) || K < 1 || K > (1LL << 30)) return IC_ERR_SIZE;
  if (nmaps < 0 || c->sweep + (uint64_t)nmaps >= (1ull << 31)) return IC_ERR_PARAM;
  for (int r = 0; r < c->replicas; ++r)
    if (!(h_T[r] > 0.0) || !std::isfinite(h_T[r])) return IC_ERR_PARAM;
  if (!d_scratch || scratch_bytes < ic_maps_scratch_bytes(c->L, K) || ((uintptr_t)d_scratch & 255) != 0) return IC_ERR_WORKSPACE;
  if (nmaps == 0) return IC_OK;
  IC_ENTER(c);
  { int rc = ensure_thresholds(c, h_T); if (rc != IC_OK) return rc; }
  MapArgs a;
  a.lattice = c->lattice; a.thr = c->d_thr; a.obs = c->d_obs; a.lat_stride = c->lat_stride;
  a.first = (int*)d_scratch; a.ia = (int*)((char*)d_scratch + align256((size_t)c->N * 4)); a.ib = a.ia + K;
  a.L = c->L; a.logL = c->logL; a.K = (int)K; a.replicas = c->replicas; a.key0 = (uint32_t)c->seed; a.key1 = (uint32_t)(c->seed >> 32);
  const double qJ = 0.25 * c->J;
  const int nb_reset = (int)std::min<long long>((c->N + 255) / 256, (long long)c->sm_count * 8);
  const unsigned nb_k = (unsigned)((K + 255) / 256);
  for (int64_t m = 0; m < nmaps; ++m) {
    a.map_index = (uint32_t)c->sweep;
    k_map_reset<<<nb_reset, 256, 0, c->stream>>>(a.first, c->N, (int)K);
    k_map_candidates<<<nb_k, 256, 0, c->stream>>>(a);
    dim3 grid(nb_k, (unsigned)c->replicas);
    if (c->layout == LAY_ROW8) k_map_update<LAY_ROW8><<<grid, 256, 0, c->stream>>>(a);
    else if (c->layout == LAY_ROW2) k_map_update<LAY_ROW2><<<grid, 256, 0, c->stream>>>(a);
    else if (c->layout == LAY_P2) k_map_update<LAY_P2><<<grid, 256, 0, c->stream>>>(a);
    else k_map_update<LAY_P16><<<grid, 256, 0, c->stream>>>(a);
    long long* trow = d_trace ? (long long*)d_trace + 6LL * c->replicas * m : nullptr;
    k_fold<<<(c->replicas + 127) / 128, 128, 0, c->stream>>>(c->d_obs, c->replicas, c->delta, c->V, qJ, trow, 0, (unsigned int*)nullptr);
    c->launches += 4;
    IC_CUDA(cudaGetLastError());
    c->sweep += 1;
  }
  return IC_OK;
}

// ---- drop observable and snapshots (Fig. 7) ------------------------------------------------------------
extern "C" size_t ic_cluster_scratch_bytes(int L) {
  if (L < 4 || L > 32768 || (L & (L - 1))) return 0;
  return (size_t)L * L * 8 + 256;
}

extern "C" int ic_largest_cluster(ic_ctx* c, int replica, int which, void* d_scratch, size_t scratch_bytes, int64_t* h_out2) {
  if (!c || !h_out2) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas || !small_index_ok(c)) return IC_ERR_SIZE;
  if (which < 0 || which > 2) return IC_ERR_PARAM;
  if (!d_scratch || scratch_bytes < ic_cluster_scratch_bytes(c->L) || ((uintptr_t)d_scratch & 255) != 0) return IC_ERR_WORKSPACE;
  IC_ENTER(c);
  int* parent = (int*)d_scratch; int* size = parent + c->N; long long* out2 = (long long*)(size + c->N);
  const LatView lat{c->lattice + (long long)replica * c->lat_stride, c->L, c->logL};
  const int nb = (int)std::min<long long>((c->N + 255) / 256, (long long)c->sm_count * 8);
  IC_CUDA(cudaMemsetAsync(out2, 0, 16, c->stream));
  if (c->layout == LAY_ROW8) k_cc_init<LAY_ROW8><<<nb, 256, 0, c->stream>>>(lat, which, parent, size);
  else if (c->layout == LAY_ROW2) k_cc_init<LAY_ROW2><<<nb, 256, 0, c->stream>>>(lat, which, parent, size);
  else if (c->layout == LAY_P2) k_cc_init<LAY_P2><<<nb, 256, 0, c->stream>>>(lat, which, parent, size);
  else k_cc_init<LAY_P16><<<nb, 256, 0, c->stream>>>(lat, which, parent, size);
  k_cc_link<<<nb, 256, 0, c->stream>>>(c->L, c->logL, parent);
  k_cc_count<<<nb, 256, 0, c->stream>>>(c->N, parent, size);
  k_cc_max<<<nb, 256, 0, c->stream>>>(c->N, size, out2);
  c->launches += 4;
  IC_CUDA(cudaGetLastError());
  long long h[2];
  IC_CUDA(cudaMemcpyAsync(h, out2, 16, cudaMemcpyDeviceToHost, c->stream));
  IC_CUDA(cudaStreamSynchronize(c->stream));
  h_out2[0] = h[0]; h_out2[1] = h[1];
  return IC_OK;
}

// Snapshot of one lattice copy as a binary PPM (P6) written from host memory: S=+1 red, S=-1 blue, sigma=+1 white, sigma=-1 dark grey.
extern "C" int ic_snapshot_ppm(ic_ctx* c, int replica, const char* path) {
  if (!c || !path) return IC_ERR_NULL;
  if (replica < 0 || replica >= c->replicas) return IC_ERR_SIZE;
  std::vector<int8_t> codes((size_t)c->N);
  int rc = ic_state(c, replica, codes.data());
  if (rc != IC_OK) return rc;
  FILE* f = fopen(path, "wb");
  if (!f) return IC_ERR_PARAM;
  fprintf(f, "P6\n%d %d\n255\n", c->L, c->L);
  static const unsigned char pal[4][3] = {{255, 255, 255}, {64, 64, 64}, {220, 30, 30}, {30, 60, 220}};
  std::vector<unsigned char> row((size_t)c->L * 3);
  for (int y = 0; y < c->L; ++y) {
    for (int x = 0; x < c->L; ++x) memcpy(&row[3 * (size_t)x], pal[codes[(size_t)y * c->L + x] & 3], 3);
    fwrite(row.data(), 1, row.size(), f);
  }
  fclose(f);
  return IC_OK;
}

// ---- ic_largest_cluster_static: the cluster count without a context, a workspace or a scratch argument ---------------------
// For callers that cannot get device memory when they need the answer (see include/ic.h: a hook inside a program that gave
// the whole HBM to its own pool, a host that forbids cudaMalloc / cudaFree because they wait for the whole device, a fixed
// memory budget).  The union-find needs parent[N] and size[N]; here both live in an array that is part of the library's
// device image: 2 x 1024 x 1024 ints = 8 MiB on every GPU that loads the library, until the process exits.
// One array per GPU, shared by every call: a call rewrites parent[0..N) and size[0..N) (k_ccs_init) before any kernel
// reads them, so what the previous call left behind does not matter; calls that overlap on the GPU race on it.
constexpr int CCS_MAX_L = IC_STATIC_CLUSTER_MAX_L;
constexpr long long CCS_MAX_N = (long long)CCS_MAX_L * CCS_MAX_L;
static __device__ __align__(256) int g_ccs_scratch[2 * CCS_MAX_N];
// On the host, `g_ccs_scratch` is NOT the device address: it is the host-side shadow variable the runtime uses as a handle.
// A kernel handed `g_ccs_scratch` from host code would write through a host address (a fault, or on systems where the GPU
// reaches host memory, silent corruption of something else).  The device address is asked for once per device, below.
constexpr int CCS_MAX_DEVICES = 64;
struct CcsDevice { int* scratch; int sm_count; };
static CcsDevice g_ccs_dev[CCS_MAX_DEVICES] = {};
static std::mutex g_ccs_mutex;

// Set-up for the calling thread's current device: device address of the array and the SM count.  Called by every
// ic_largest_cluster_static; only the first call per device talks to the runtime.  No allocation.
static int ccs_setup(CcsDevice* out) {
  int dev = -1;
  IC_CUDA(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_ccs_mutex);
  const bool cached = dev >= 0 && dev < CCS_MAX_DEVICES;
  if (cached && g_ccs_dev[dev].scratch) { *out = g_ccs_dev[dev]; return IC_OK; }
  CcsDevice d{nullptr, 0};
  IC_CUDA(cudaGetSymbolAddress((void**)&d.scratch, g_ccs_scratch));   // the copy of the array on the CURRENT device
  IC_CUDA(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
  if (!d.scratch || ((uintptr_t)d.scratch & 255) != 0 || d.sm_count < 1) return cuda_fail(cudaErrorInvalidSymbol, "address of the built-in scratch array");
  if (cached) g_ccs_dev[dev] = d;
  *out = d;
  return IC_OK;
}

// parent[i] = i for sites inside the selection, -1 outside; size[i] = 0; the caller's two outputs start at zero.
// Everything the later kernels read is written here first: the array still holds the previous call's forest.
__global__ void k_ccs_init(const int8_t* __restrict__ codes, int N, int which, int* __restrict__ parent, int* __restrict__ size,
                           long long* __restrict__ out2) {
  if (blockIdx.x == 0 && threadIdx.x == 0) { out2[0] = 0; out2[1] = 0; }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
    parent[i] = cc_inside(codes[i] & 3, which) ? i : -1;
    size[i] = 0;
  }
}

static bool ccs_gpu_can_read(const void* p) {      // false for ordinary (pageable, unregistered) host memory
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type != cudaMemoryTypeUnregistered;
}

extern "C" int ic_largest_cluster_static(const int8_t* d_codes, int L, int which, int64_t* d_out2, void* cuda_stream) {
  if (!d_codes || !d_out2) return IC_ERR_NULL;
  if (L < 4 || (L & (L - 1)) != 0) return IC_ERR_SIZE;
  if (L > CCS_MAX_L) return IC_ERR_STATIC_MAX;
  if (which < 0 || which > 2) return IC_ERR_PARAM;
  if (!ccs_gpu_can_read(d_codes) || !ccs_gpu_can_read(d_out2)) return IC_ERR_PARAM;
  CcsDevice d;
  { int rc = ccs_setup(&d); if (rc != IC_OK) return rc; }
  const int N = L * L;
  int logL = 0; while ((1 << logL) < L) ++logL;
  int* parent = d.scratch; int* size = d.scratch + N;      // the first 8 N bytes of the array, whatever CCS_MAX_N is
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const int nb = (int)std::min<long long>((N + 255) / 256, (long long)d.sm_count * 8);
  k_ccs_init<<<nb, 256, 0, stream>>>(d_codes, N, which, parent, size, (long long*)d_out2);
  k_cc_link<<<nb, 256, 0, stream>>>(L, logL, parent);
  k_cc_count<<<nb, 256, 0, stream>>>(N, parent, size);
  k_cc_max<<<nb, 256, 0, stream>>>(N, size, (long long*)d_out2);
  IC_CUDA(cudaGetLastError());
  return IC_OK;
}

extern "C" int ic_thresholds(ic_ctx* c, double T, uint32_t* h_out) {
  if (!c || !h_out) return IC_ERR_NULL;
  if (!(T > 0.0) || !std::isfinite(T)) return IC_ERR_PARAM;
  std::vector<uint32_t> tmp(THR_STRIDE);
  build_thresholds(c, T, tmp.data());
  memcpy(h_out, tmp.data(), sizeof(uint32_t) * N_CLASSES);
  return IC_OK;
}

extern "C" int ic_schedule(ic_ctx* c, uint64_t sweep, int32_t* out4) {
  if (!c || !out4) return IC_ERR_NULL;
  if (sweep >= (1ull << 31)) return IC_ERR_PARAM;
  schedule_params(c->L, c->seed, sweep, out4);
  return IC_OK;
}

extern "C" int64_t ic_sweep_count(const ic_ctx* c) { return c ? (int64_t)c->sweep : -1; }
extern "C" int64_t ic_charge(const ic_ctx* c) { return c ? (int64_t)c->Q : 0; }
extern "C" int ic_kernel_family(const ic_ctx* c) { return c ? c->last_family : -1; }
extern "C" int64_t ic_launch_count(const ic_ctx* c) { return c ? (int64_t)c->launches : -1; }

extern "C" int ic_set_variant(ic_ctx* c, int variant) {
  if (!c) return IC_ERR_NULL;
  if (variant < 0 || variant > 6) return IC_ERR_PARAM;
  if (variant == 6 && !resvec_ok(c)) return IC_ERR_PARAM;
  if (variant == 5 && !coop_ok(c)) return IC_ERR_PARAM;
  if (variant == 4 && c->L > RES_MAX_L) return IC_ERR_PARAM;
  if (variant == 2 && !tiled_ok(c)) return IC_ERR_PARAM;
  if (variant == 3 && !staged_ok(c)) return IC_ERR_PARAM;
  c->variant = variant;
  return IC_OK;
}

extern "C" int ic_set_max_blocks(ic_ctx* c, int max_blocks) {
  if (!c) return IC_ERR_NULL;
  if (max_blocks < 0) return IC_ERR_PARAM;
  c->max_blocks = max_blocks;
  return IC_OK;
}

extern "C" const char* ic_strerror(int code) {
  switch (code) {
    case IC_OK: return "ok";
    case IC_ERR_NULL: return "a required pointer is NULL";
    case IC_ERR_SIZE: return "invalid size: L must be a power of two in [4, 65536], replicas >= 1, bits_per_site 8 or 2, replica in range";
    case IC_ERR_PARAM: return "invalid parameter: |n| <= 1, finite Delta, V, J, T > 0, nsweeps >= 0, sweep counter < 2^31";
    case IC_ERR_WORKSPACE: return "workspace is NULL, too small (see ic_workspace_bytes) or not 256-byte aligned";
    case IC_ERR_CHARGE: return "state rejected: a code outside 0..3 or sum S != Q";
    case IC_ERR_CUDA: return g_cuda_msg;
    case IC_ERR_STATIC_MAX: return "ic_largest_cluster_static: L is larger than IC_STATIC_CLUSTER_MAX_L (1024), the lattice does not fit the scratch array built into the library; use ic_largest_cluster with scratch memory of your own";
    default: return "unknown error code";
  }
}
