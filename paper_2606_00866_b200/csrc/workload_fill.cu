// workload_fill.cu -- libmori_workload.so: CUDA twin of workload.page_content (the seeded,
// counter-based page-content generator) plus a checker.  INPUT GENERATION ONLY: nothing here is
// part of the hot path and libmori.so does not link it.  Must match the numpy version bit for
// bit (integer hash, one IEEE multiply, round-to-nearest-even to bf16; no fast-math).
#include <cuda_runtime.h>
#include <cstdint>

namespace {

__host__ __device__ inline uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}

__device__ inline uint32_t f32_to_bf16_bits(float f) {
  uint32_t u = __float_as_uint(f);
  return (u + 0x7FFFu + ((u >> 16) & 1u)) >> 16;
}

__device__ inline uint32_t word_of(uint64_t key, uint32_t layer, uint32_t w) {
  const uint64_t h = splitmix64(key ^ (((uint64_t)layer << 32) + w));
  uint32_t out = 0;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    int s = 0;
#pragma unroll
    for (int b = 0; b < 4; ++b) s += (int)((h >> (8 * (4 * half + b))) & 0xFF);
    const float f = __fmul_rn((float)(s - 510), 1.0f / 147.8f);
    out |= f32_to_bf16_bits(f) << (16 * half);
  }
  return out;
}

// pool [L][P][chunk]; page j: key keys[j], physical page pages[j].  grid.x strides over
// (page, layer) pairs; threads over the words of the chunk.
template <bool kCheck>
__global__ void fill_or_check(uint32_t* pool, long long P, int L, int words, const uint64_t* keys,
                              const int32_t* pages, long long n, long long page_stride_words,
                              long long layer_stride_words, unsigned long long* mismatches) {
  unsigned long long bad = 0;
  for (long long pl = blockIdx.x; pl < n * L; pl += gridDim.x) {
    const long long j = pl / L;
    const int l = (int)(pl - j * L);
    uint32_t* dst = pool + (long long)pages[j] * page_stride_words + (long long)l * layer_stride_words;
    const uint64_t key = keys[j];
    for (int w = threadIdx.x; w < words; w += blockDim.x) {
      const uint32_t v = word_of(key, (uint32_t)l, (uint32_t)w);
      if (kCheck) bad += dst[w] != v; else dst[w] = v;
    }
  }
  if (kCheck && bad) atomicAdd(mismatches, bad);
}

}  // namespace

extern "C" {

// Pool layout: word address of (layer l, page g) = g*page_stride_words + l*layer_stride_words.
//   device pool [L][P][chunk]:  page_stride = words, layer_stride = P*words
//   host arena  [S][L][chunk]:  page_stride = L*words, layer_stride = words
int wl_fill_pages(void* pool, long long P, int L, int chunk_bytes, const uint64_t* keys_dev,
                  const int32_t* pages_dev, long long n, int arena_layout, void* stream) {
  if (n == 0) return 0;
  const int words = chunk_bytes / 4;
  const long long ps = arena_layout ? (long long)L * words : words;
  const long long ls = arena_layout ? words : P * (long long)words;
  const int grid = (int)(n * L < 148 * 16 ? n * L : 148 * 16);
  fill_or_check<false><<<grid, 256, 0, (cudaStream_t)stream>>>((uint32_t*)pool, P, L, words, keys_dev,
                                                                pages_dev, n, ps, ls, nullptr);
  return (int)cudaGetLastError();
}

int wl_check_pages(const void* pool, long long P, int L, int chunk_bytes, const uint64_t* keys_dev,
                   const int32_t* pages_dev, long long n, int arena_layout,
                   unsigned long long* mismatches_dev, void* stream) {
  if (n == 0) return 0;
  const int words = chunk_bytes / 4;
  const long long ps = arena_layout ? (long long)L * words : words;
  const long long ls = arena_layout ? words : P * (long long)words;
  const int grid = (int)(n * L < 148 * 16 ? n * L : 148 * 16);
  fill_or_check<true><<<grid, 256, 0, (cudaStream_t)stream>>>((uint32_t*)pool, P, L, words, keys_dev,
                                                               pages_dev, n, ps, ls, mismatches_dev);
  return (int)cudaGetLastError();
}

}  // extern "C"
