// a10_rans.cu -- NEXT-3, the entropy stage behind the residual transform: static rANS over independent
// chunks of a symbol stream ("TPC rANS Encoding"; readings P57..P60 in DESIGN.md; tpc_rans_encode /
// tpc_rans_decode in include/tpc_track.h).
//
// A chunk is the unit of parallelism: rANS is serial in its state, so one thread codes one chunk (512 symbols by
// default: 35 000 threads per residual stream of the bench batch) with the frequency and cumulative tables in shared
// memory.  Encoding runs backwards through the chunk and pushes its 16-bit words downwards from the end of the
// chunk's slot in a scratch buffer (a step emits at most one word, so 4 + 2 * chunk bytes bound a chunk); a scan over
// the chunk sizes and a warp-per-chunk copy pack the slots into the payload.  Integer arithmetic only: the bytes are
// the oracle's.
//   count  : symbol histogram (shared-memory bins) + escapes per chunk
//   table  : P58 normalisation, one CTA
//   scan   : exclusive offsets of the per-chunk escape counts / byte sizes, one CTA
//   encode : thread per chunk -> scratch slots, sizes; escapes to their place
//   pack   : warp per chunk, slot -> payload
//   decode : thread per chunk, symbol by binary search over the cumulative table
#include <mutex>

#include "tpc_internal.cuh"

namespace {

constexpr int RANS_THREADS = 256;
constexpr uint32_t RANS_M = 65536u;
constexpr int RANS_MAX_BITS = 12;   // tables of 2^12 entries in shared memory

template <typename T>
__device__ __forceinline__ int32_t value_at(const void* v, int64_t i) { return (int32_t)((const T*)v)[i]; }

__device__ __forceinline__ uint32_t symbol_of(int32_t v, int32_t half) {   // P57
  return (v > -half && v < half) ? (uint32_t)(v + half) : 0u;
}

template <typename T>
__global__ void __launch_bounds__(RANS_THREADS)
rans_count_kernel(const void* __restrict__ values, int64_t n, int32_t bits, int32_t chunk, uint32_t* __restrict__ hist,
                  uint32_t* __restrict__ esc_cnt) {
  __shared__ uint32_t s_hist[1 << RANS_MAX_BITS];
  const int A = 1 << bits, half = A >> 1;
  for (int s = threadIdx.x; s < A; s += blockDim.x) s_hist[s] = 0;
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const uint32_t s = symbol_of(value_at<T>(values, i), half);
    atomicAdd(&s_hist[s], 1u);
    if (s == 0) atomicAdd(&esc_cnt[i / chunk], 1u);
  }
  __syncthreads();
  for (int s = threadIdx.x; s < A; s += blockDim.x)
    if (s_hist[s]) atomicAdd(&hist[s], s_hist[s]);
}

// P58: f_s = 1 + floor(n_s (M - K) / N) for the symbols that occur, the remainder to the most frequent (the smallest
// among equals); cum[s] = sum of f below s.  One CTA.
__global__ void __launch_bounds__(1024)
rans_table_kernel(int32_t bits, int64_t n, const uint32_t* __restrict__ hist, uint32_t* __restrict__ freq,
                  uint32_t* __restrict__ cum) {
  __shared__ uint32_t s_f[1 << RANS_MAX_BITS];
  __shared__ uint32_t s_K, s_sum;
  __shared__ unsigned long long s_top;
  const int A = 1 << bits;
  if (threadIdx.x == 0) { s_K = 0; s_sum = 0; s_top = 0; }
  __syncthreads();
  for (int s = threadIdx.x; s < A; s += blockDim.x)
    if (hist[s]) {
      atomicAdd(&s_K, 1u);
      atomicMax(&s_top, ((unsigned long long)hist[s] << 16) | (unsigned long long)(0xFFFF - s));
    }
  __syncthreads();
  const uint32_t K = s_K;
  for (int s = threadIdx.x; s < A; s += blockDim.x) {
    const uint32_t c = hist[s];
    const uint32_t f = c ? 1u + (uint32_t)(((unsigned long long)c * (RANS_M - K)) / (unsigned long long)n) : 0u;
    s_f[s] = f;
    if (f) atomicAdd(&s_sum, f);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (n > 0) s_f[0xFFFF - (int)(s_top & 0xFFFF)] += RANS_M - s_sum;
    uint32_t run = 0;
    for (int s = 0; s < A; ++s) {
      cum[s] = run;
      run += s_f[s];
    }
    cum[A] = run;
  }
  __syncthreads();
  for (int s = threadIdx.x; s < A; s += blockDim.x) freq[s] = s_f[s];
}

// off[0 .. m] = exclusive prefix sums of cnt[0 .. m-1] (off[m] = the total, also written to *total64).  One CTA.
__global__ void __launch_bounds__(1024)
rans_scan_kernel(const uint32_t* __restrict__ cnt, int64_t m, uint32_t* __restrict__ off, int64_t* __restrict__ total64) {
  __shared__ uint32_t wsum[33];
  uint32_t carry = 0;
  for (int64_t base = 0; base < m; base += blockDim.x) {
    const int64_t i = base + threadIdx.x;
    const uint32_t v = i < m ? cnt[i] : 0u;
    uint32_t tot;
    const uint32_t ex = block_excl_scan(v, wsum, &tot);
    if (i < m) off[i] = carry + ex;
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    off[m] = carry;
    *total64 = (int64_t)carry;
  }
}

// P59 / P60, one thread per chunk.  slot c of `scratch` is [c * stride, (c + 1) * stride), stride = 4 + 2 * chunk.
template <typename T>
__global__ void __launch_bounds__(RANS_THREADS)
rans_encode_kernel(const void* __restrict__ values, int64_t n, int32_t bits, int32_t chunk, int64_t n_chunks,
                   const uint32_t* __restrict__ freq, const uint32_t* __restrict__ cum,
                   const uint32_t* __restrict__ esc_off, int64_t esc_cap, uint8_t* __restrict__ scratch,
                   uint32_t* __restrict__ size, int32_t* __restrict__ escapes) {
  __shared__ uint32_t s_f[1 << RANS_MAX_BITS], s_c[1 << RANS_MAX_BITS];
  const int A = 1 << bits, half = A >> 1;
  for (int s = threadIdx.x; s < A; s += blockDim.x) {
    s_f[s] = freq[s];
    s_c[s] = cum[s];
  }
  __syncthreads();
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_chunks) return;
  const int64_t i0 = c * chunk, i1 = min(n, i0 + (int64_t)chunk);
  const size_t stride = 4 + 2 * (size_t)chunk;
  uint16_t* const end = (uint16_t*)(scratch + (size_t)(c + 1) * stride);
  uint16_t* wp = end;
  int64_t e = (int64_t)esc_off[c + 1];   // escapes of the chunk are written backwards too: stream order in the end
  uint32_t x = RANS_M;
  for (int64_t i = i1 - 1; i >= i0; --i) {
    const int32_t v = value_at<T>(values, i);
    const uint32_t s = symbol_of(v, half);
    if (s == 0) {
      --e;
      if (e < esc_cap) escapes[e] = v;
    }
    const uint32_t f = s_f[s];
    if ((unsigned long long)x >= ((unsigned long long)f << 16)) {
      *--wp = (uint16_t)(x & 0xFFFFu);
      x >>= 16;
    }
    x = ((x / f) << 16) + (x % f) + s_c[s];
  }
  *--wp = (uint16_t)(x >> 16);       // the state, little endian: low half first
  *--wp = (uint16_t)(x & 0xFFFFu);
  size[c] = (uint32_t)((end - wp) * 2);
}

// slot -> payload, one warp per chunk, 16-bit units (sizes and offsets are even).
__global__ void __launch_bounds__(RANS_THREADS)
rans_pack_kernel(int32_t chunk, int64_t n_chunks, const uint8_t* __restrict__ scratch,
                 const uint32_t* __restrict__ chunk_off, int64_t payload_cap, uint8_t* __restrict__ payload) {
  const int lane = threadIdx.x & 31;
  const int64_t warps = (int64_t)gridDim.x * (blockDim.x >> 5);
  const size_t stride = 4 + 2 * (size_t)chunk;
  for (int64_t c = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); c < n_chunks; c += warps) {
    const uint32_t a = chunk_off[c], b = chunk_off[c + 1];
    if ((int64_t)b > payload_cap) continue;   // overflow: flagged by the caller's counts, nothing written beyond
    const uint16_t* src = (const uint16_t*)(scratch + (size_t)(c + 1) * stride - (b - a));
    uint16_t* dst = (uint16_t*)(payload + a);
    for (uint32_t k = lane; k < (b - a) / 2; k += 32) dst[k] = src[k];
  }
}

__global__ void rans_counts_kernel(int64_t n_chunks, int64_t payload_cap, int64_t esc_cap, int64_t* __restrict__ counts) {
  // counts[0] = payload bytes and counts[1] = escapes were written by the scans
  counts[2] = n_chunks;
  counts[3] = (counts[0] > payload_cap ? 1 : 0) | (counts[1] > esc_cap ? 2 : 0);
}

template <typename T>
__global__ void __launch_bounds__(RANS_THREADS)
rans_decode_kernel(int64_t n, int32_t bits, int32_t chunk, int64_t n_chunks, const uint32_t* __restrict__ freq,
                   const uint32_t* __restrict__ chunk_off, const uint32_t* __restrict__ esc_off,
                   const uint8_t* __restrict__ payload, const int32_t* __restrict__ escapes, void* __restrict__ values) {
  __shared__ uint32_t s_f[1 << RANS_MAX_BITS], s_c[(1 << RANS_MAX_BITS) + 1];
  __shared__ uint32_t wsum[33];
  const int A = 1 << bits, half = A >> 1;
  // cumulative table from the frequencies: block scan over tiles of blockDim.x symbols
  uint32_t carry = 0;
  for (int base = 0; base < A; base += blockDim.x) {
    const int s = base + threadIdx.x;
    const uint32_t f = s < A ? freq[s] : 0u;
    uint32_t tot;
    const uint32_t ex = block_excl_scan(f, wsum, &tot);
    if (s < A) {
      s_f[s] = f;
      s_c[s] = carry + ex;
    }
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) s_c[A] = carry;
  __syncthreads();
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_chunks) return;
  const int64_t i0 = c * chunk, i1 = min(n, i0 + (int64_t)chunk);
  const uint16_t* in = (const uint16_t*)(payload + chunk_off[c]);
  uint32_t x = (uint32_t)in[0] | ((uint32_t)in[1] << 16);
  in += 2;
  int64_t e = esc_off[c];
  for (int64_t i = i0; i < i1; ++i) {
    const uint32_t slot = x & 0xFFFFu;
    int lo = 0, hi = A;   // the last s with cum[s] <= slot: symbols that do not occur have empty intervals
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (s_c[mid] <= slot) lo = mid; else hi = mid;
    }
    const uint32_t s = (uint32_t)lo;
    x = s_f[s] * (x >> 16) + slot - s_c[s];
    if (x < RANS_M) x = (x << 16) | (uint32_t)(*in++);
    const int32_t v = s == 0 ? escapes[e++] : (int32_t)s - half;
    ((T*)values)[i] = (T)v;
  }
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

size_t rans_scratch_bytes(int64_t n, int32_t chunk, int32_t bits) {
  const int64_t n_chunks = (n + chunk - 1) / chunk;
  // slots | hist[A] | cum[A + 1] | esc_cnt[n_chunks] | size[n_chunks], each part 16-byte aligned
  return align_up((size_t)n_chunks * (4 + 2 * (size_t)chunk), 16) + align_up(((size_t)1 << bits) * 4, 16) +
         align_up((((size_t)1 << bits) + 1) * 4, 16) + 2 * align_up((size_t)(n_chunks + 1) * 4, 16);
}

cudaError_t launch_a10_rans_encode(const tpc_tracker* t, const void* values, int32_t value_bytes, int64_t n,
                                   int32_t bits, int32_t chunk, const tpc_rans_stream_t* out, cudaStream_t st) {
  const int A = 1 << bits;
  const int64_t n_chunks = (n + chunk - 1) / chunk;
  char* p = (char*)t->rans_scratch;
  uint8_t* slots = (uint8_t*)p;        p += align_up((size_t)n_chunks * (4 + 2 * (size_t)chunk), 16);
  uint32_t* hist = (uint32_t*)p;       p += align_up((size_t)A * 4, 16);
  uint32_t* cum = (uint32_t*)p;        p += align_up(((size_t)A + 1) * 4, 16);
  uint32_t* esc_cnt = (uint32_t*)p;    p += align_up((size_t)(n_chunks + 1) * 4, 16);
  uint32_t* size = (uint32_t*)p;
  cudaError_t e = cudaMemsetAsync(hist, 0, (size_t)A * 4, st);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(esc_cnt, 0, (size_t)(n_chunks + 1) * 4, st);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(out->counts, 0, 4 * sizeof(int64_t), st);
  if (e != cudaSuccess) return e;
  const int grid_el = (int)std::min<int64_t>((n + RANS_THREADS - 1) / RANS_THREADS, (int64_t)t->a4_sms * 8);
  const int grid_ch = (int)((n_chunks + RANS_THREADS - 1) / RANS_THREADS);
  if (n > 0) {
    if (value_bytes == 1)
      rans_count_kernel<uint8_t><<<grid_el, RANS_THREADS, 0, st>>>(values, n, bits, chunk, hist, esc_cnt);
    else
      rans_count_kernel<int32_t><<<grid_el, RANS_THREADS, 0, st>>>(values, n, bits, chunk, hist, esc_cnt);
  }
  rans_table_kernel<<<1, 1024, 0, st>>>(bits, n, hist, out->freq, cum);
  rans_scan_kernel<<<1, 1024, 0, st>>>(esc_cnt, n_chunks, out->esc_off, out->counts + 1);
  if (n > 0) {
    if (value_bytes == 1)
      rans_encode_kernel<uint8_t><<<grid_ch, RANS_THREADS, 0, st>>>(values, n, bits, chunk, n_chunks, out->freq, cum,
                                                                     out->esc_off, out->escape_capacity, slots, size,
                                                                     out->escapes);
    else
      rans_encode_kernel<int32_t><<<grid_ch, RANS_THREADS, 0, st>>>(values, n, bits, chunk, n_chunks, out->freq, cum,
                                                                     out->esc_off, out->escape_capacity, slots, size,
                                                                     out->escapes);
  }
  rans_scan_kernel<<<1, 1024, 0, st>>>(size, n_chunks, out->chunk_off, out->counts);
  if (n > 0)
    rans_pack_kernel<<<t->a4_sms * 8, RANS_THREADS, 0, st>>>(chunk, n_chunks, slots, out->chunk_off,
                                                            out->payload_capacity, out->payload);
  rans_counts_kernel<<<1, 1, 0, st>>>(n_chunks, out->payload_capacity, out->escape_capacity, out->counts);
  return cudaGetLastError();
}

cudaError_t launch_a10_rans_decode(const tpc_tracker* t, const tpc_rans_stream_t* in, int64_t n, int32_t bits,
                                   int32_t chunk, void* values, int32_t value_bytes, cudaStream_t st) {
  (void)t;
  const int64_t n_chunks = (n + chunk - 1) / chunk;
  if (n == 0) return cudaSuccess;
  const int grid_ch = (int)((n_chunks + RANS_THREADS - 1) / RANS_THREADS);
  if (value_bytes == 1)
    rans_decode_kernel<uint8_t><<<grid_ch, RANS_THREADS, 0, st>>>(n, bits, chunk, n_chunks, in->freq, in->chunk_off,
                                                                   in->esc_off, in->payload, in->escapes, values);
  else
    rans_decode_kernel<int32_t><<<grid_ch, RANS_THREADS, 0, st>>>(n, bits, chunk, n_chunks, in->freq, in->chunk_off,
                                                                   in->esc_off, in->payload, in->escapes, values);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------
// tpc_rans_encode_static (include/tpc_track.h): the encoder for callers that must not allocate.  Same kernels, same
// scratch layout; the scratch is this array, part of the library image on every GPU that loads it.  In host code the
// name g_rans_static_scratch is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress,
// once per device, with that device current, and that pointer is what the kernels get.
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_rans_static_scratch[TPC_RANS_STATIC_SCRATCH_BYTES];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
void* g_static_ptr[STATIC_MAX_DEVICES];   // device address of the array, per device ordinal (NULL: not looked up yet)
int g_static_sms[STATIC_MAX_DEVICES];

// the launch sequence of launch_a10_rans_encode on a scratch pointer of the caller's
cudaError_t enqueue_rans_encode(char* scratch, int sms, const void* values, int32_t value_bytes, int64_t n, int32_t bits,
                                int32_t chunk, const tpc_rans_stream_t* out, cudaStream_t st) {
  const int A = 1 << bits;
  const int64_t n_chunks = (n + chunk - 1) / chunk;
  char* p = scratch;
  uint8_t* slots = (uint8_t*)p;        p += align_up((size_t)n_chunks * (4 + 2 * (size_t)chunk), 16);
  uint32_t* hist = (uint32_t*)p;       p += align_up((size_t)A * 4, 16);
  uint32_t* cum = (uint32_t*)p;        p += align_up(((size_t)A + 1) * 4, 16);
  uint32_t* esc_cnt = (uint32_t*)p;    p += align_up((size_t)(n_chunks + 1) * 4, 16);
  uint32_t* size = (uint32_t*)p;
  // the array holds the previous call's contents: the histogram and the escape counts are accumulated into, so they
  // start at zero; cum, size and the slots are written before they are read
  cudaError_t e = cudaMemsetAsync(hist, 0, (size_t)A * 4, st);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(esc_cnt, 0, (size_t)(n_chunks + 1) * 4, st);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(out->counts, 0, 4 * sizeof(int64_t), st);
  if (e != cudaSuccess) return e;
  const int grid_el = (int)std::min<int64_t>((n + RANS_THREADS - 1) / RANS_THREADS, (int64_t)sms * 8);
  const int grid_ch = (int)((n_chunks + RANS_THREADS - 1) / RANS_THREADS);
  if (n > 0) {
    if (value_bytes == 1)
      rans_count_kernel<uint8_t><<<grid_el, RANS_THREADS, 0, st>>>(values, n, bits, chunk, hist, esc_cnt);
    else
      rans_count_kernel<int32_t><<<grid_el, RANS_THREADS, 0, st>>>(values, n, bits, chunk, hist, esc_cnt);
  }
  rans_table_kernel<<<1, 1024, 0, st>>>(bits, n, hist, out->freq, cum);
  rans_scan_kernel<<<1, 1024, 0, st>>>(esc_cnt, n_chunks, out->esc_off, out->counts + 1);
  if (n > 0) {
    if (value_bytes == 1)
      rans_encode_kernel<uint8_t><<<grid_ch, RANS_THREADS, 0, st>>>(values, n, bits, chunk, n_chunks, out->freq, cum,
                                                                     out->esc_off, out->escape_capacity, slots, size,
                                                                     out->escapes);
    else
      rans_encode_kernel<int32_t><<<grid_ch, RANS_THREADS, 0, st>>>(values, n, bits, chunk, n_chunks, out->freq, cum,
                                                                     out->esc_off, out->escape_capacity, slots, size,
                                                                     out->escapes);
  }
  rans_scan_kernel<<<1, 1024, 0, st>>>(size, n_chunks, out->chunk_off, out->counts);
  if (n > 0)
    rans_pack_kernel<<<sms * 8, RANS_THREADS, 0, st>>>(chunk, n_chunks, slots, out->chunk_off, out->payload_capacity,
                                                       out->payload);
  rans_counts_kernel<<<1, 1, 0, st>>>(n_chunks, out->payload_capacity, out->escape_capacity, out->counts);
  return cudaGetLastError();
}

}  // namespace


extern "C" {
#pragma GCC visibility push(default)

int tpc_rans_encode_static(const void* values, int32_t value_bytes, int64_t n, int32_t alphabet_bits, int32_t chunk,
                           void* stream, const tpc_rans_stream_t* out) {
  if (!out || n < 0 || n >= ((int64_t)1 << 31) || (value_bytes != 1 && value_bytes != 4)) return TPC_ERR_ARG;
  if (alphabet_bits < 1 || alphabet_bits > RANS_MAX_BITS || chunk < 1 || chunk > 65535) return TPC_ERR_ARG;
  if (!out->freq || !out->chunk_off || !out->esc_off || !out->counts || out->payload_capacity < 0 ||
      out->escape_capacity < 0)
    return TPC_ERR_ARG;
  if (n > 0 && (!values || (out->payload_capacity > 0 && !out->payload) || (out->escape_capacity > 0 && !out->escapes)))
    return TPC_ERR_ARG;
  if (rans_scratch_bytes(n, chunk, alphabet_bits) > (size_t)TPC_RANS_STATIC_SCRATCH_BYTES) return TPC_ERR_STATIC_SCRATCH;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return TPC_ERR_CUDA;
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return TPC_ERR_ARG;
  char* scratch = nullptr;
  int sms = 0;
  {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {   // once per device, with that device current
      void* p = nullptr;
      if (cudaGetSymbolAddress(&p, g_rans_static_scratch) != cudaSuccess || !p) return TPC_ERR_CUDA;
      int count = 0;
      if (cudaDeviceGetAttribute(&count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || count <= 0)
        return TPC_ERR_CUDA;
      g_static_sms[dev] = count;
      g_static_ptr[dev] = p;
    }
    scratch = (char*)g_static_ptr[dev];
    sms = g_static_sms[dev];
  }
  if (enqueue_rans_encode(scratch, sms, values, value_bytes, n, alphabet_bits, chunk, out, (cudaStream_t)stream) !=
      cudaSuccess)
    return TPC_ERR_CUDA;
  return TPC_OK;
}

#pragma GCC visibility pop
}  // extern "C"
