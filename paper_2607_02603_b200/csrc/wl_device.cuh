// Device-side building blocks shared by the kernels of the CUDA path (sm_100a).
// Nothing in here is used by, or taken from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wl {

typedef unsigned long long u64;
typedef unsigned int u32;

// device scalar block (u64 each): counters the kernels keep between launches; kScalLog.. = colour count per queued round
enum {
  kScalNew = 0,        // new ids handed out by the running relabel step
  kScalErr = 1,        // validation error bits
  kScalCanon = 2,      // number of blocks found by the canonicalisation
  kScalActive = 3,     // rows kept by the last compaction
  kScalActiveDeg = 4,  // their out-degree sum
  kScalHub = 5,        // hub chunks
  kScalActiveHub = 6,  // hub rows kept by the last compaction
  kScalK = 7,          // current number of colours
  kScalTicket = 8,     // CTAs that finished relabel_finish_kernel
  kScalErrAux = 9,     // validation error bits written on the side stream
  kScalRowTicket = 10, // row-group ticket of spmv_rows32_tag_kernel
  kScalFrontier = 11,  // worklist regime: largest |L| of a round since the host last reset it
  kScalLog = 16,
  kNumScal = 64
};

// error bits written by device-side validation
constexpr u32 kErrRowPtr = 1u, kErrCol = 2u, kErrRowSum = 4u, kErrInit = 8u;

// ---- weight bijection (readings Q4/Q5; Alg. 1 lines 3-4) -------------------------------
// mix is a bijection of Z/2^64: xor-shifts and odd multipliers are invertible.  M1/M2/G are
// floor(frac(sqrt 2) 2^64)|1, floor(frac(sqrt 3) 2^64)|1, floor(frac(golden ratio) 2^64)|1.
constexpr u64 kM1 = 0x6a09e667f3bcc909ull;
constexpr u64 kM2 = 0xbb67ae8584caa73bull;
constexpr u64 kG = 0x9e3779b97f4a7c15ull;

__host__ __device__ __forceinline__ u64 mix64(u64 x) {
  x ^= x >> 32;
  x *= kM1;
  x ^= x >> 29;
  x *= kM2;
  x ^= x >> 32;
  return x;
}
__host__ __device__ __forceinline__ u64 round_key(u64 seed, u64 stream, u64 round) {
  return mix64(mix64(mix64(seed + kG) + stream) + round);
}
// weight of dense colour id c under `key`
__host__ __device__ __forceinline__ u64 weight_of(u64 key, u64 c) { return mix64(c + key); }

// The ring is Z/2^q (Alg. 1 "precision parameter q >= 1", L109-L110; L100).  q = 64 unless the caller asks for a smaller ring
// (wl_options.ring_bits): every z is then reduced to its low q bits wherever it is compared or keyed.  Sums and products commute
// with the reduction, so masking at the point of use is Algorithm 1 over Z/2^q exactly.  A small q makes the collisions of
// Lemma 1 (L418) frequent enough to be counted (tests/test_gpu_collisions.py); Theorem 1's guarantee needs q >= 64.
__host__ __device__ __forceinline__ u64 ring_mask(int q) { return (q <= 0 || q >= 64) ? ~0ull : ((1ull << q) - 1); }

// ---- 128-bit hash slot and its atomics -------------------------------------------------------------------------------
// slot = { y : 64 | colour : 32 | x : 32 }.  EMPTY = all ones.  x = new dense id once assigned.
struct __align__(16) Slot {
  u64 y;
  u64 cx;  // low 32 bits: old colour, high 32 bits: x
};
constexpr u64 kEmpty = ~0ull;

__device__ __forceinline__ Slot cas128(Slot* p, Slot cmp, Slot val) {
  Slot old;
  asm volatile(
      "{\n\t.reg .b128 c, v, o;\n\t"
      "mov.b128 c, {%2, %3};\n\t"
      "mov.b128 v, {%4, %5};\n\t"
      "atom.global.relaxed.gpu.cas.b128 o, [%6], c, v;\n\t"
      "mov.b128 {%0, %1}, o;\n\t}"
      : "=l"(old.y), "=l"(old.cx)
      : "l"(cmp.y), "l"(cmp.cx), "l"(val.y), "l"(val.cx), "l"(p)
      : "memory");
  return old;
}
// 16-byte load that bypasses L1 (table contents change during the kernel)
__device__ __forceinline__ Slot load_slot(const Slot* p) {
  Slot s;
  asm volatile("ld.global.cg.v2.u64 {%0, %1}, [%2];" : "=l"(s.y), "=l"(s.cx) : "l"(p) : "memory");
  return s;
}
__device__ __forceinline__ void store_slot(Slot* p, u64 y, u64 cx) {
  asm volatile("st.global.cg.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(y), "l"(cx) : "memory");
}

__device__ __forceinline__ u64 slot_hash(u32 c, u64 y) {
  u64 h = (y ^ (y >> 31)) * kG + (u64)c * kM1;
  return h ^ (h >> 29);
}

// streaming loads: column indices are read exactly once per round
__device__ __forceinline__ int ld_stream_i32(const int* p) {
  int v;
  asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ u32 ld_stream_u32(const u32* p) {
  u32 v;
  asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}

// no-return 64-bit add at L2 (RED.E.ADD.64): sums in Z/2^64 are order independent, so any schedule is bit exact
__device__ __forceinline__ void red_add_u64(u64* p, u64 v) { atomicAdd(p, v); }

// block-wide exclusive scan of a 0/1 flag; returns rank, *total = number of set flags in the block
template <int THREADS>
__device__ __forceinline__ int block_rank(bool flag, int* total) {
  __shared__ int s_warp[THREADS / 32 + 1];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned b = __ballot_sync(0xffffffffu, flag);
  const int in_warp = __popc(b & ((1u << lane) - 1));
  if (lane == 0) s_warp[wid] = __popc(b);
  __syncthreads();
  if (threadIdx.x == 0) {
    int run = 0;
    for (int w = 0; w < THREADS / 32; ++w) {
      int t = s_warp[w];
      s_warp[w] = run;
      run += t;
    }
    s_warp[THREADS / 32] = run;
  }
  __syncthreads();
  *total = s_warp[THREADS / 32];
  const int r = s_warp[wid] + in_warp;
  __syncthreads();  // s_warp may be reused by a later call
  return r;
}

}  // namespace wl
