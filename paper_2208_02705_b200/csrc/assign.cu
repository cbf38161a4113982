// r360 -- Algorithm 1, stage II (text :157): geometry-aware assignment of the occupied
// voxels to n tiny networks.
//
//   s <- S / n ;  for k <- 1..n:  pop an unassigned voxel with the minimum coordinate as the anchor,
//                                 search s-1 nearest unassigned neighbours, assign these s voxels to network k
//
// Readings S1-S4: the first S mod n networks take one voxel more; "minimum coordinate" = smallest
// linear index; "nearest" = squared centre distance in metres, binary32, d2 = ((dx*sx)^2 + (dy*sy)^2) + (dz*sz)^2
// with every operation rounded; ties go to the smaller linear index.  So the candidates of one iteration are
// totally ordered by the 57-bit key (bits of d2) << 25 | position (position in the ascending list of occupied
// voxels), and "the s-1 nearest" are the keys up to the (s-1)-th smallest one.  That key is found by a radix
// select, most significant digit first (12, 12, 12, 12, 9 bits): one histogram pass over the unassigned voxels
// per digit, no sort and no tie handling.  The n iterations are sequential by definition (each removes
// voxels from the next one's candidates); one iteration is 12 small launches, captured once in a CUDA graph.
#include <cstring>
#include <limits>
#include <new>
#include <vector>

#include "scene.h"

namespace {

constexpr int kPasses = 5;
constexpr int kDigitBits[kPasses] = {12, 12, 12, 12, 9};
constexpr int kDigitShift[kPasses] = {45, 33, 21, 9, 0};
constexpr int kPosBits = 25;
constexpr int kBins = 4096;

struct AssignState {
  unsigned long long prefix;   // digits of the wanted key chosen so far; the whole key after the last pass
  uint32_t rank;               // rank (1-based) of the wanted key among the candidates that match the prefix
  uint32_t need;               // s - 1 of this iteration (0: nothing to search)
  uint32_t cursor;             // no unassigned voxel lies below this position
  uint32_t k;                  // network of this iteration
  uint32_t q, r;               // S = n*q + r
  float ax, ay, az;            // anchor voxel index, as floats
  uint32_t failed;             // an iteration found no anchor or no digit (cannot happen for n <= S)
};

struct Voxels {
  const ushort4* coord;        // [S] voxel index (x, y, z) of the occupied voxels, ascending linear index
  int32_t* label;              // [S] -1 = unassigned
  uint32_t S;
  float sx, sy, sz;            // voxel size (reading C)
};

__device__ __forceinline__ unsigned long long make_key(const Voxels& v, const AssignState& st, uint32_t i) {
  const ushort4 c = v.coord[i];
  // reading S3: exact integer differences, then one rounding per operation
  const float dx = __fmul_rn((float)c.x - st.ax, v.sx);
  const float dy = __fmul_rn((float)c.y - st.ay, v.sy);
  const float dz = __fmul_rn((float)c.z - st.az, v.sz);
  const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
  return ((unsigned long long)__float_as_uint(d2) << kPosBits) | i;
}

// pop the unassigned voxel with the minimum coordinate (reading S2) and open iteration k
__global__ void __launch_bounds__(1024) k_anchor(Voxels v, AssignState* st) {
  __shared__ uint32_t found;
  uint32_t pos = st->cursor;
  if (threadIdx.x == 0) found = 0xFFFFFFFFu;
  __syncthreads();
  while (pos < v.S) {
    const uint32_t i = pos + threadIdx.x;
    if (i < v.S && v.label[i] < 0) atomicMin(&found, i);
    __syncthreads();
    // every thread takes the window's result into a register and the block meets again before anyone starts the
    // next window's atomicMin: a thread lagging behind this read could otherwise see a value of a later window
    // (ADVICE round 1), and all threads leave the loop in the same iteration
    const uint32_t f = found;
    __syncthreads();
    if (f != 0xFFFFFFFFu) break;
    pos += blockDim.x;
  }
  if (threadIdx.x == 0) {
    const uint32_t k = st->k;
    if (found == 0xFFFFFFFFu) {
      st->failed = 1;
      st->need = 0;
    } else {
      const ushort4 c = v.coord[found];
      v.label[found] = (int32_t)k;
      st->ax = (float)c.x; st->ay = (float)c.y; st->az = (float)c.z;
      st->cursor = found + 1;
      const uint32_t size = st->q + (k < st->r ? 1u : 0u);   // reading S1
      st->need = size - 1;
      st->rank = size - 1;
      st->prefix = 0;
    }
  }
}

// histogram of digit `pass` of the keys of the unassigned voxels whose higher digits equal the prefix
template <int PASS>
__global__ void __launch_bounds__(256) k_hist(Voxels v, const AssignState* st, uint32_t* hist) {
  __shared__ uint32_t sh[kBins];
  const AssignState s = *st;
  if (s.need == 0) return;
  constexpr int bits = kDigitBits[PASS], shift = kDigitShift[PASS];
  for (int b = threadIdx.x; b < (1 << bits); b += blockDim.x) sh[b] = 0;
  __syncthreads();
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < v.S; i += gridDim.x * blockDim.x) {
    if (v.label[i] >= 0) continue;
    const unsigned long long key = make_key(v, s, i);
    if ((key >> (shift + bits)) != s.prefix) continue;
    atomicAdd(&sh[(uint32_t)(key >> shift) & ((1u << bits) - 1)], 1u);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < (1 << bits); b += blockDim.x)
    if (sh[b]) atomicAdd(&hist[b], sh[b]);
}

// the digit whose bin holds the wanted rank; the histogram is cleared for the next iteration
template <int PASS>
__global__ void __launch_bounds__(1024) k_pick(AssignState* st, uint32_t* hist) {
  __shared__ uint32_t warp_tot[33];
  if (st->need == 0) return;
  constexpr int bits = kDigitBits[PASS];
  constexpr int per = kBins / 1024;                            // 4 bins per thread
  const uint32_t rank = st->rank;
  uint32_t c[per], sum = 0;
#pragma unroll
  for (int u = 0; u < per; ++u) {
    const int b = threadIdx.x * per + u;
    c[u] = b < (1 << bits) ? hist[b] : 0u;
    if (b < (1 << bits)) hist[b] = 0;
    sum += c[u];
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += y;
  }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = warp_tot[lane], wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += y;
    }
    warp_tot[lane] = wi - w;
    if (lane == 31) warp_tot[32] = wi;
  }
  __syncthreads();
  uint32_t below = warp_tot[wid] + incl - sum;                 // candidates in the bins before this thread's
#pragma unroll
  for (int u = 0; u < per; ++u) {
    if (below < rank && rank <= below + c[u]) {                // exactly one (thread, u) when rank <= total
      st->prefix = (st->prefix << bits) | (unsigned long long)(threadIdx.x * per + u);
      st->rank = rank - below;
    }
    below += c[u];
  }
  if (threadIdx.x == 0 && warp_tot[32] < rank) st->failed = 1;
}

// every unassigned voxel whose key is not above the selected one joins network k; next iteration
__global__ void __launch_bounds__(256) k_take(Voxels v, AssignState* st_rw) {
  const AssignState s = *st_rw;
  if (s.need != 0) {
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < v.S; i += gridDim.x * blockDim.x)
      if (v.label[i] < 0 && make_key(v, s, i) <= s.prefix) v.label[i] = (int32_t)s.k;
  }
}
__global__ void k_next(AssignState* st) { st->k += 1; }

}  // namespace

extern "C" r360_status r360_assign_subfields(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                             const uint8_t* occupancy, uint8_t occ_threshold, int32_t n,
                                             int32_t* labels_out) {
  if (!dims || !box_min || !box_max || !occupancy || !labels_out || n < 1 || occ_threshold < 1)
    return R360_ERR_INVALID_ARG;
  for (int a = 0; a < 3; ++a)
    if (dims[a] < 1 || dims[a] > 65535 || !(box_max[a] > box_min[a])) return R360_ERR_INVALID_ARG;
  const long long N = (long long)dims[0] * dims[1] * dims[2];
  std::vector<ushort4> coord;
  std::vector<long long> lin;
  std::vector<int32_t> lab;               // (every host allocation inside the try: no exception crosses the C ABI)
  try {
    for (long long vox = 0; vox < N; ++vox) {
      labels_out[vox] = -1;
      if (occupancy[vox] < occ_threshold) continue;
      coord.push_back(make_ushort4((unsigned short)(vox % dims[0]), (unsigned short)((vox / dims[0]) % dims[1]),
                                   (unsigned short)(vox / ((long long)dims[0] * dims[1])), 0));
      lin.push_back(vox);
    }
    lab.resize(coord.size());
  } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
  const size_t S = coord.size();
  if ((size_t)n > S || S >= (1ull << kPosBits)) return R360_ERR_INVALID_ARG;

  Voxels v{};
  v.S = (uint32_t)S;
  float vs[3];
  for (int a = 0; a < 3; ++a) {                                // voxel size exactly as the renderer computes it
    volatile float ext = box_max[a] - box_min[a];
    vs[a] = ext / (float)dims[a];
  }
  v.sx = vs[0]; v.sy = vs[1]; v.sz = vs[2];
  ushort4* d_coord = nullptr;
  int32_t* d_label = nullptr;
  AssignState* d_st = nullptr;
  uint32_t* d_hist = nullptr;
  cudaStream_t stream = nullptr;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  r360_status rc = R360_OK;
  auto fail = [&](cudaError_t e, const char* what) { rc = r360_cuda_fail(e, what); };
#define A_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { fail(e_, #call); goto done; } } while (0)
  {
    AssignState h{};
    h.q = (uint32_t)(S / (size_t)n);
    h.r = (uint32_t)(S % (size_t)n);
    A_CUDA(cudaStreamCreateWithFlags(&stream, cudaStreamNonBlocking));
    A_CUDA(cudaMalloc(&d_coord, S * sizeof(ushort4)));
    A_CUDA(cudaMalloc(&d_label, S * sizeof(int32_t)));
    A_CUDA(cudaMalloc(&d_st, sizeof(AssignState)));
    A_CUDA(cudaMalloc(&d_hist, kPasses * kBins * sizeof(uint32_t)));
    A_CUDA(cudaMemcpyAsync(d_coord, coord.data(), S * sizeof(ushort4), cudaMemcpyHostToDevice, stream));
    A_CUDA(cudaMemsetAsync(d_label, 0xFF, S * sizeof(int32_t), stream));
    A_CUDA(cudaMemsetAsync(d_hist, 0, kPasses * kBins * sizeof(uint32_t), stream));
    A_CUDA(cudaMemcpyAsync(d_st, &h, sizeof(h), cudaMemcpyHostToDevice, stream));
    v.coord = d_coord;
    v.label = d_label;
    int n_sms = 148, dev = 0;
    A_CUDA(cudaGetDevice(&dev));
    A_CUDA(cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev));
    int blocks = (int)((S + 255) / 256);
    if (blocks > n_sms * 8) blocks = n_sms * 8;
    // one iteration = 12 launches; captured once, replayed n times
    A_CUDA(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
    k_anchor<<<1, 1024, 0, stream>>>(v, d_st);
    k_hist<0><<<blocks, 256, 0, stream>>>(v, d_st, d_hist + 0 * kBins);
    k_pick<0><<<1, 1024, 0, stream>>>(d_st, d_hist + 0 * kBins);
    k_hist<1><<<blocks, 256, 0, stream>>>(v, d_st, d_hist + 1 * kBins);
    k_pick<1><<<1, 1024, 0, stream>>>(d_st, d_hist + 1 * kBins);
    k_hist<2><<<blocks, 256, 0, stream>>>(v, d_st, d_hist + 2 * kBins);
    k_pick<2><<<1, 1024, 0, stream>>>(d_st, d_hist + 2 * kBins);
    k_hist<3><<<blocks, 256, 0, stream>>>(v, d_st, d_hist + 3 * kBins);
    k_pick<3><<<1, 1024, 0, stream>>>(d_st, d_hist + 3 * kBins);
    k_hist<4><<<blocks, 256, 0, stream>>>(v, d_st, d_hist + 4 * kBins);
    k_pick<4><<<1, 1024, 0, stream>>>(d_st, d_hist + 4 * kBins);
    k_take<<<blocks, 256, 0, stream>>>(v, d_st);
    k_next<<<1, 1, 0, stream>>>(d_st);
    A_CUDA(cudaStreamEndCapture(stream, &graph));
    A_CUDA(cudaGraphInstantiate(&exec, graph, 0));
    for (int k = 0; k < n; ++k) A_CUDA(cudaGraphLaunch(exec, stream));
    A_CUDA(cudaMemcpyAsync(lab.data(), d_label, S * sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    A_CUDA(cudaMemcpyAsync(&h, d_st, sizeof(h), cudaMemcpyDeviceToHost, stream));
    A_CUDA(cudaStreamSynchronize(stream));
    if (h.failed) { rc = R360_ERR_CUDA; goto done; }
    for (size_t i = 0; i < S; ++i) labels_out[lin[i]] = lab[i];
  }
done:
#undef A_CUDA
  if (exec) cudaGraphExecDestroy(exec);
  if (graph) cudaGraphDestroy(graph);
  cudaFree(d_coord); cudaFree(d_label); cudaFree(d_st); cudaFree(d_hist);
  if (stream) cudaStreamDestroy(stream);
  return rc;
}
