// pack.cu -- A0: one-time packing of a catalogue into the segmented (CSR) layout that replaces the
// paper's padded (N_events, N_pix, N_samples) tensor (its own future work).
// Stable sort of samples by (event, row) -- ties keep input order, so the answer is unique and integer --
// then event offsets, the distinct rows of each event and the start of each (event, row) run.
// The sort itself is the CUB library radix sort (a library primitive on a one-time, non-hot step);
// everything else is plain kernels.
#include <cub/block/block_scan.cuh>
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <math_constants.h>

#include "gwc_internal.h"

namespace gwc {

namespace {

__global__ void pack_keys_kernel(int64_t n, int64_t n_events, const int32_t* __restrict__ ev,
                                 const int32_t* __restrict__ row, uint64_t* __restrict__ keys,
                                 int64_t* __restrict__ idx, int* flag) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int32_t e = ev[k], r = row[k];
  if (e < 0 || e >= n_events || r < 0) atomicOr(flag, 2);
  keys[k] = ((uint64_t)(uint32_t)e << 32) | (uint64_t)(uint32_t)r;
  idx[k] = k;
}

// ev_sample_off[i] = first sorted position whose event id is >= i
__global__ void pack_event_off_kernel(int64_t n, int64_t n_events, const uint64_t* __restrict__ keys,
                                      int64_t* __restrict__ ev_sample_off) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i > n_events) return;
  const uint64_t key = (uint64_t)i << 32;
  int64_t lo = 0, hi = n;
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (keys[mid] < key) lo = mid + 1; else hi = mid;
  }
  ev_sample_off[i] = lo;
}

__global__ void pack_heads_kernel(int64_t n, const uint64_t* __restrict__ keys, int64_t* __restrict__ head) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  head[k] = (k == 0 || keys[k] != keys[k - 1]) ? 1 : 0;
}

// pos = exclusive scan of head.  Scatter run starts; the last thread writes the count and the end sentinel.
__global__ void pack_runs_kernel(int64_t n, const uint64_t* __restrict__ keys, const int64_t* __restrict__ head,
                                 const int64_t* __restrict__ pos, int32_t* __restrict__ ev_pix_rows,
                                 int64_t* __restrict__ pix_sample_off, int64_t* __restrict__ n_pixrefs) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  if (head[k]) {
    ev_pix_rows[pos[k]] = (int32_t)(uint32_t)(keys[k] & 0xffffffffu);
    pix_sample_off[pos[k]] = k;
  }
  if (k == n - 1) {
    const int64_t np = pos[k] + head[k];
    *n_pixrefs = np;
    pix_sample_off[np] = n;
  }
}

__global__ void pack_pix_off_kernel(int64_t n, int64_t n_events, const int64_t* __restrict__ ev_sample_off,
                                    const int64_t* __restrict__ pos, const int64_t* __restrict__ n_pixrefs,
                                    int64_t* __restrict__ ev_pix_off) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i > n_events) return;
  const int64_t s = ev_sample_off[i];
  ev_pix_off[i] = (i == n_events || s >= n) ? *n_pixrefs : pos[s];
}

__global__ void pack_empty_kernel(int64_t n_events, int64_t* ev_sample_off, int64_t* ev_pix_off,
                                  int64_t* pix_sample_off, int64_t* n_pixrefs) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i <= n_events) {
    ev_sample_off[i] = 0;
    ev_pix_off[i] = 0;
  }
  if (i == 0) {
    pix_sample_off[0] = 0;
    *n_pixrefs = 0;
  }
}

// ---- per-pixel sample cap (R31) ---------------------------------------------------
// upper half of splitmix64's output function applied to seed + (index + 1) * golden ratio
__device__ __forceinline__ uint32_t cap_hash32(uint64_t seed, uint64_t index) {
  uint64_t z = seed + (index + 1ULL) * 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  z = z ^ (z >> 31);
  return (uint32_t)(z >> 32);
}

// key of packed position k = (its pixel, hash of its original sample index); value = k
__global__ void cap_keys_kernel(int64_t n, int64_t n_pix, const int64_t* __restrict__ perm,
                                const int64_t* __restrict__ pix_sample_off, uint64_t seed, uint64_t* __restrict__ keys,
                                int64_t* __restrict__ vals) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  int64_t lo = 0, hi = n_pix;  // largest j with pix_sample_off[j] <= k
  while (hi - lo > 1) {
    const int64_t mid = (lo + hi) >> 1;
    if (pix_sample_off[mid] <= k) lo = mid; else hi = mid;
  }
  keys[k] = ((uint64_t)lo << 32) | (uint64_t)cap_hash32(seed, (uint64_t)perm[k]);
  vals[k] = k;
}

// after the stable sort the samples of a pixel are in (hash, packed position) order: the first `cap` are kept
__global__ void cap_flags_kernel(int64_t n, const uint64_t* __restrict__ keys_sorted,
                                 const int64_t* __restrict__ vals_sorted, const int64_t* __restrict__ pix_sample_off,
                                 int64_t cap, int64_t* __restrict__ keep) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t j = (int64_t)(keys_sorted[i] >> 32);
  keep[vals_sorted[i]] = (i - pix_sample_off[j] < cap) ? 1 : 0;
}

__global__ void cap_compact_kernel(int64_t n, const int64_t* __restrict__ perm_in, const int64_t* __restrict__ keep,
                                   const int64_t* __restrict__ newpos, int64_t* __restrict__ perm_out,
                                   int64_t* __restrict__ n_kept) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  if (keep[k]) perm_out[newpos[k]] = perm_in[k];
  if (k == n - 1) *n_kept = newpos[k] + keep[k];
}

// offsets of the kept samples, in place (each thread reads its own old value)
__global__ void cap_offsets_kernel(int64_t n, int64_t m, int64_t* __restrict__ off, const int64_t* __restrict__ newpos,
                                   const int64_t* __restrict__ n_kept) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i > m) return;
  const int64_t o = off[i];
  off[i] = o >= n ? *n_kept : newpos[o];
}

size_t a256(size_t x) { return (x + 255) & ~(size_t)255; }

size_t cub_temp_bytes(int64_t n) {
  size_t a = 0, b = 0;
  cub::DeviceRadixSort::SortPairs(nullptr, a, (const uint64_t*)nullptr, (uint64_t*)nullptr, (const int64_t*)nullptr,
                                  (int64_t*)nullptr, n);
  cub::DeviceScan::ExclusiveSum(nullptr, b, (const int64_t*)nullptr, (int64_t*)nullptr, n);
  return a > b ? a : b;
}

}  // namespace

size_t pack_scratch_bytes(int64_t n_samples, int64_t n_events) {
  (void)n_events;
  const size_t n = (size_t)(n_samples > 0 ? n_samples : 1);
  return 4 * a256(8 * n) + a256(cub_temp_bytes((int64_t)n)) + 256;
}

int launch_pack(int64_t n, int64_t n_events, const int32_t* d_event_id, const int32_t* d_row, int64_t* d_perm,
                int64_t* d_ev_sample_off, int64_t* d_ev_pix_off, int32_t* d_ev_pix_rows, int64_t* d_pix_sample_off,
                int64_t* d_n_pixrefs, int* d_flag, void* scratch, size_t scratch_bytes, cudaStream_t s) {
  int launches = 0;
  const unsigned be = (unsigned)((n_events + 1 + 255) / 256);
  if (n == 0) {
    pack_empty_kernel<<<be, 256, 0, s>>>(n_events, d_ev_sample_off, d_ev_pix_off, d_pix_sample_off, d_n_pixrefs);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
  }
  unsigned char* base = (unsigned char*)scratch;
  uint64_t* keys = (uint64_t*)base;            base += a256(8 * (size_t)n);
  uint64_t* keys_sorted = (uint64_t*)base;     base += a256(8 * (size_t)n);
  int64_t* idx = (int64_t*)base;               base += a256(8 * (size_t)n);
  int64_t* head = (int64_t*)base;              base += a256(8 * (size_t)n);
  void* temp = base;
  size_t temp_bytes = scratch_bytes - (size_t)(base - (unsigned char*)scratch);
  const unsigned bn = (unsigned)((n + 255) / 256);
  pack_keys_kernel<<<bn, 256, 0, s>>>(n, n_events, d_event_id, d_row, keys, idx, d_flag);
  ++launches;
  int end_bit = 32;
  while (end_bit < 64 && ((uint64_t)n_events >> (end_bit - 32)) != 0) ++end_bit;
  if (cub::DeviceRadixSort::SortPairs(temp, temp_bytes, keys, keys_sorted, idx, d_perm, n, 0, end_bit, s) !=
      cudaSuccess)
    return -1;
  launches += 8;  // radix passes (library; approximate count)
  pack_event_off_kernel<<<be, 256, 0, s>>>(n, n_events, keys_sorted, d_ev_sample_off);
  pack_heads_kernel<<<bn, 256, 0, s>>>(n, keys_sorted, head);
  int64_t* pos = idx;  // the unsorted index array is free again
  temp_bytes = scratch_bytes - (size_t)(base - (unsigned char*)scratch);
  if (cub::DeviceScan::ExclusiveSum(temp, temp_bytes, head, pos, n, s) != cudaSuccess) return -1;
  pack_runs_kernel<<<bn, 256, 0, s>>>(n, keys_sorted, head, pos, d_ev_pix_rows, d_pix_sample_off, d_n_pixrefs);
  pack_pix_off_kernel<<<be, 256, 0, s>>>(n, n_events, d_ev_sample_off, pos, d_n_pixrefs, d_ev_pix_off);
  launches += 6;
  return cudaGetLastError() == cudaSuccess ? launches : -1;
}

size_t cap_scratch_bytes(int64_t n_samples) {
  const size_t n = (size_t)(n_samples > 0 ? n_samples : 1);
  return 6 * a256(8 * n) + a256(cub_temp_bytes((int64_t)n)) + 256;
}

// Per-pixel sample cap on a packed catalogue: rewrites the two offset arrays for the kept samples, writes the kept
// entries of perm_in to perm_out (packed order preserved) and their number to d_n_kept.
int launch_cap_pixels(int64_t n, int64_t n_events, int64_t n_pix, const int64_t* d_perm_in, int64_t* d_ev_sample_off,
                      int64_t* d_pix_sample_off, int64_t cap, uint64_t seed, int64_t* d_perm_out, int64_t* d_n_kept,
                      void* scratch, size_t scratch_bytes, cudaStream_t s) {
  if (n == 0) {
    if (cudaMemsetAsync(d_n_kept, 0, sizeof(int64_t), s) != cudaSuccess) return -1;
    return 0;
  }
  unsigned char* base = (unsigned char*)scratch;
  uint64_t* keys = (uint64_t*)base;            base += a256(8 * (size_t)n);
  uint64_t* keys_sorted = (uint64_t*)base;     base += a256(8 * (size_t)n);
  int64_t* vals = (int64_t*)base;              base += a256(8 * (size_t)n);
  int64_t* vals_sorted = (int64_t*)base;       base += a256(8 * (size_t)n);
  int64_t* keep = (int64_t*)base;              base += a256(8 * (size_t)n);
  int64_t* newpos = (int64_t*)base;            base += a256(8 * (size_t)n);
  void* temp = base;
  size_t temp_bytes = scratch_bytes - (size_t)(base - (unsigned char*)scratch);
  const unsigned bn = (unsigned)((n + 255) / 256);
  cap_keys_kernel<<<bn, 256, 0, s>>>(n, n_pix, d_perm_in, d_pix_sample_off, seed, keys, vals);
  int end_bit = 33;
  while (end_bit < 64 && ((uint64_t)n_pix >> (end_bit - 32)) != 0) ++end_bit;
  if (cub::DeviceRadixSort::SortPairs(temp, temp_bytes, keys, keys_sorted, vals, vals_sorted, n, 0, end_bit, s) !=
      cudaSuccess)
    return -1;
  cap_flags_kernel<<<bn, 256, 0, s>>>(n, keys_sorted, vals_sorted, d_pix_sample_off, cap, keep);
  temp_bytes = scratch_bytes - (size_t)(base - (unsigned char*)scratch);
  if (cub::DeviceScan::ExclusiveSum(temp, temp_bytes, keep, newpos, n, s) != cudaSuccess) return -1;
  cap_compact_kernel<<<bn, 256, 0, s>>>(n, d_perm_in, keep, newpos, d_perm_out, d_n_kept);
  cap_offsets_kernel<<<(unsigned)((n_events + 1 + 255) / 256), 256, 0, s>>>(n, n_events, d_ev_sample_off, newpos, d_n_kept);
  cap_offsets_kernel<<<(unsigned)((n_pix + 1 + 255) / 256), 256, 0, s>>>(n, n_pix, d_pix_sample_off, newpos, d_n_kept);
  return cudaGetLastError() == cudaSuccess ? 14 : -1;  // 5 kernels + the library's radix and scan passes (approximate)
}

}  // namespace gwc

// ---- pixel-aligned layout of the prepared samples (pixel-cut mode of the fused kernel) ---------------------------------
// The fused kernel's lanes own two consecutive samples.  In the copy made here every pixel (a maximal run of equal
// sample_row inside a segment, R25) starts at an even position and has an even length: a run of odd length
// is followed by one dead slot (dLc = NaN, same row).  Then a lane never straddles two pixels, which is what makes
// the per-(theta, pixel) sums of Eq. 8 a plain segmented scan over lanes (reweight.cu).  theta-independent: built
// once per catalogue call (kept between calls with gwc_cache_catalogue).  One CTA per segment walks its samples in
// order, 256 at a time: run start of every sample by a max-scan of the head positions, pad flag at odd-length tails,
// running count of pads = the sample's shift.
namespace gwc {
namespace {

constexpr int PAD_THREADS = 256;
struct PadSrc {
  const double *dLc, *m1z, *m2z, *L1, *Q, *P;
  const int32_t* row;
};
struct PadDst {
  double *dLc, *m1z, *m2z, *L1, *Q, *P;
  int32_t* row;
};

template <bool SCATTER>
__global__ void __launch_bounds__(PAD_THREADS) pixpad_kernel(const int64_t* __restrict__ seg_off,
                                                              const int32_t* __restrict__ row,
                                                              int64_t* __restrict__ seg_pads,          // !SCATTER: out
                                                              const int64_t* __restrict__ seg_off_pad,  // SCATTER: in
                                                              PadSrc src, PadDst dst) {
  typedef cub::BlockScan<long long, PAD_THREADS> Scan;
  __shared__ typename Scan::TempStorage tmp;
  __shared__ long long s_head, s_pads;
  const int seg = blockIdx.x, tid = threadIdx.x;
  const int64_t s0 = seg_off[seg], s1 = seg_off[seg + 1];
  if (tid == 0) {
    s_head = s0;
    s_pads = 0;
  }
  __syncthreads();
  const int64_t base_out = SCATTER ? seg_off_pad[seg] : 0;
  for (int64_t base = s0; base < s1; base += PAD_THREADS) {
    const int64_t k = base + tid;
    const bool in = k < s1;
    const int32_t r = in ? row[k] : 0;
    const bool head = in && (k == s0 || row[k - 1] != r);
    const bool tail = in && (k + 1 == s1 || row[k + 1] != r);
    long long start;   // first sample of the run that holds k
    Scan(tmp).InclusiveScan(head ? (long long)k : -1LL, start, cub::Max());
    __syncthreads();
    const long long carry_head = s_head, carry_pads = s_pads;
    start = start > carry_head ? start : carry_head;
    const bool pad = tail && (((k - start) & 1) == 0);   // odd length
    long long shift, total;
    Scan(tmp).ExclusiveSum(pad ? 1LL : 0LL, shift, total);
    __syncthreads();
    if (SCATTER && in) {
      const int64_t o = base_out + (k - s0) + carry_pads + shift;
      dst.dLc[o] = src.dLc[k];
      dst.m1z[o] = src.m1z[k];
      dst.m2z[o] = src.m2z[k];
      dst.L1[o] = src.L1[k];
      dst.Q[o] = src.Q[k];
      dst.P[o] = src.P[k];
      dst.row[o] = r;
      if (pad) {
        dst.dLc[o + 1] = CUDART_NAN;
        dst.m1z[o + 1] = 1.0;
        dst.m2z[o + 1] = 1.0;
        dst.L1[o + 1] = 0.0;
        dst.Q[o + 1] = 0.0;
        dst.P[o + 1] = 0.0;
        dst.row[o + 1] = r;
      }
    }
    if (tid == PAD_THREADS - 1) {   // (slots past the end repeat the last run start)
      s_head = start;
      s_pads = carry_pads + total;
    }
    __syncthreads();
  }
  if (!SCATTER && tid == 0) seg_pads[seg] = s_pads;
}

// seg_off_pad[i] = seg_off[i] + pads of the segments before i (single CTA, in order)
__global__ void __launch_bounds__(PAD_THREADS) pixpad_offsets_kernel(const int64_t* __restrict__ seg_off,
                                                                      const int64_t* __restrict__ seg_pads,
                                                                      int64_t n_seg, int64_t* __restrict__ seg_off_pad) {
  typedef cub::BlockScan<long long, PAD_THREADS> Scan;
  __shared__ typename Scan::TempStorage tmp;
  __shared__ long long s_carry;
  const int tid = threadIdx.x;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  for (int64_t base = 0; base <= n_seg; base += PAD_THREADS) {
    const int64_t i = base + tid;
    long long excl, total;
    Scan(tmp).ExclusiveSum(i < n_seg ? (long long)seg_pads[i] : 0LL, excl, total);
    __syncthreads();
    const long long carry = s_carry;
    if (i <= n_seg) seg_off_pad[i] = seg_off[i] + carry + excl;
    __syncthreads();
    if (tid == 0) s_carry = carry + total;
    __syncthreads();
  }
}

}  // namespace

int launch_pixpad_count(const int64_t* d_seg_off, int64_t n_seg, const int32_t* d_row, int64_t* d_seg_pads,
                        int64_t* d_seg_off_pad, cudaStream_t s) {
  if (n_seg <= 0) return 0;
  PadSrc src = {};
  PadDst dst = {};
  pixpad_kernel<false><<<(unsigned)n_seg, PAD_THREADS, 0, s>>>(d_seg_off, d_row, d_seg_pads, nullptr, src, dst);
  pixpad_offsets_kernel<<<1, PAD_THREADS, 0, s>>>(d_seg_off, d_seg_pads, n_seg, d_seg_off_pad);
  return cudaGetLastError() == cudaSuccess ? 2 : -1;
}

int launch_pixpad_scatter(const int64_t* d_seg_off, int64_t n_seg, const int64_t* d_seg_off_pad, const double* dLc,
                          const double* m1z, const double* m2z, const double* L1, const double* Q, const double* P,
                          const int32_t* row, double* o_dLc, double* o_m1z, double* o_m2z, double* o_L1, double* o_Q,
                          double* o_P, int32_t* o_row, cudaStream_t s) {
  if (n_seg <= 0) return 0;
  PadSrc src = {dLc, m1z, m2z, L1, Q, P, row};
  PadDst dst = {o_dLc, o_m1z, o_m2z, o_L1, o_Q, o_P, o_row};
  pixpad_kernel<true><<<(unsigned)n_seg, PAD_THREADS, 0, s>>>(d_seg_off, row, nullptr, d_seg_off_pad, src, dst);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace gwc

// ---- injections in order of d_L (selection term) ----------------------------------------------------------------------
// The selection sum does not depend on the order of the injections (beyond rounding), and in order of d_L whole
// warps fall outside a theta's table together and skip it: one radix sort of the d_L bit patterns (positive doubles
// order like their bits; invalid values end up anywhere, they are dead) and a gather of the four arrays, once per
// injection set (kept between calls with gwc_cache_catalogue).
namespace gwc {
namespace {
__global__ void injsort_keys_kernel(int64_t n, const double* __restrict__ dL, uint64_t* __restrict__ keys,
                                    int64_t* __restrict__ idx) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  keys[k] = (uint64_t)__double_as_longlong(dL[k]);
  idx[k] = k;
}
__global__ void injsort_gather_kernel(int64_t n, const int64_t* __restrict__ perm, const double* __restrict__ a,
                                      const double* __restrict__ b, const double* __restrict__ c,
                                      const double* __restrict__ d, double* __restrict__ oa, double* __restrict__ ob,
                                      double* __restrict__ oc, double* __restrict__ od) {
  const int64_t k = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int64_t j = perm[k];
  oa[k] = a[j];
  ob[k] = b[j];
  oc[k] = c[j];
  od[k] = d[j];
}
}  // namespace

size_t injsort_scratch_bytes(int64_t n) {
  const size_t m = (size_t)(n > 0 ? n : 1);
  return 4 * a256(8 * m) + a256(cub_temp_bytes((int64_t)m)) + 256;
}

int launch_injsort(int64_t n, const double* dL, const double* m1z, const double* m2z, const double* lp, double* o_dL,
                   double* o_m1z, double* o_m2z, double* o_lp, void* scratch, size_t scratch_bytes, cudaStream_t s) {
  if (n <= 0) return 0;
  unsigned char* base = (unsigned char*)scratch;
  uint64_t* keys = (uint64_t*)base;          base += a256(8 * (size_t)n);
  uint64_t* keys_sorted = (uint64_t*)base;   base += a256(8 * (size_t)n);
  int64_t* idx = (int64_t*)base;             base += a256(8 * (size_t)n);
  int64_t* perm = (int64_t*)base;            base += a256(8 * (size_t)n);
  size_t temp = scratch_bytes - (size_t)(base - (unsigned char*)scratch);
  const unsigned blocks = (unsigned)((n + 255) / 256);
  injsort_keys_kernel<<<blocks, 256, 0, s>>>(n, dL, keys, idx);
  if (cub::DeviceRadixSort::SortPairs(base, temp, keys, keys_sorted, idx, perm, n, 0, 64, s) != cudaSuccess) return -1;
  injsort_gather_kernel<<<blocks, 256, 0, s>>>(n, perm, dL, m1z, m2z, lp, o_dL, o_m1z, o_m2z, o_lp);
  return cudaGetLastError() == cudaSuccess ? 3 : -1;
}

}  // namespace gwc
