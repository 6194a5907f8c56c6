// Deep-round regime of S5: worklist refinement.  Algorithm 1 recomputes every row in every round (L113-
// L125); on graphs that need hundreds of rounds (the 2048^2 grid: 1024) almost nothing changes per round.  Once the
// loop is past its first rounds, the engine keeps ONE weight function (a fixed key) so that y_i stays valid as long as no
// out-neighbour of i changes colour, and per round touches only
//   D = in-neighbours of the nodes that changed colour in the previous round  (they are the only rows whose y can change),
//   L = the nodes of D whose y did change                                       (they are the only nodes that can move).
// A node of L leaves its block for the block of the exact key (old colour, new y).  If every member of a block leaves, one of
// the resulting groups inherits the old id, so ids stay dense and a block that moves as a whole does not change at all.
// The partition after every round is the one Algorithm 1 produces (same trajectory, same fixed point); the union bound of
// Theorem 1 is over the weights of the colours alive in a round, which are uniform and distinct under a fixed key as well.
// Needs the in-neighbour lists (a transposed CSR built on the device when the regime starts).
#pragma once
#include "wl_kernels.cuh"

namespace wl {

// device scalars of the deep regime (u64 each), inside the workspace
enum {
  kDeepChanged0 = 0,  // |C| of even rounds
  kDeepChanged1 = 1,  // |C| of odd rounds
  kDeepLeavers0 = 2,  // |L| of even rounds
  kDeepLeavers1 = 3,  // |L| of odd rounds
  kDeepSlots = 4,     // slots claimed this round
  kDeepNew = 5,       // fresh ids handed out this round
  kNumDeep = 8
};

// ---- warp-aggregated list appends and keyed counters (a single word would otherwise take one atomic per item) -----------
// every lane of the warp must call; returns the list position of a lane with flag set
__device__ __forceinline__ u64 warp_append(bool flag, u64* __restrict__ counter) {
  const unsigned bal = __ballot_sync(0xffffffffu, flag);
  if (bal == 0) return 0;
  const int lane = threadIdx.x & 31, leader = __ffs(bal) - 1;
  u64 base = 0;
  if (lane == leader) base = atomicAdd(counter, (u64)__popc(bal));
  base = __shfl_sync(0xffffffffu, base, leader);
  return base + (u64)__popc(bal & ((1u << lane) - 1));
}
// arr[key] += sign * (number of active lanes with that key); every lane of the warp must call
__device__ __forceinline__ void warp_count_by_key(bool active, int key, int* __restrict__ arr, int sign) {
  const unsigned peers = __match_any_sync(0xffffffffu, active ? key : -1);
  if (active && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(arr + key, sign * __popc(peers));
}

// ---- transposed CSR (in-neighbour lists), built once ------------------------------------------------------------------
__global__ void deep_indegree_kernel(int64_t m, const int* __restrict__ col, int* __restrict__ indeg) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < m; p += stride) atomicAdd(indeg + col[p], 1);
}

// one warp per source row: in-neighbour lists are filled in any order (cursor[j] counts down from indeg[j])
__global__ void __launch_bounds__(256)
deep_fill_kernel(int64_t n, const int64_t* __restrict__ row_ptr, const int* __restrict__ col,
                 const int64_t* __restrict__ tp_ptr, int* __restrict__ cursor, int* __restrict__ tp_src) {
  const int lane = threadIdx.x & 31;
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (i >= n) return;
  const int64_t a = row_ptr[i], b = row_ptr[i + 1];
  for (int64_t p = a + lane; p < b; p += 32) {
    const int j = col[p];
    const int slot = atomicSub(cursor + j, 1) - 1;
    tp_src[tp_ptr[j] + slot] = (int)i;
  }
}

// block sizes, warp-aggregated (the giant block of a grid would otherwise serialise millions of adds on one word)
__global__ void deep_sizes_kernel(int64_t n, const int* __restrict__ colour, int* __restrict__ size) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = i < n;
  const int c = valid ? colour[i] : -1;
  const unsigned peers = __match_any_sync(0xffffffffu, c);
  if (valid && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(size + c, __popc(peers));
}

// ---- one round ---------------------------------------------------------------------------------------------------------
// Two kernels per round: deep_front_kernel (the rows with a changed out-neighbour get their new y; those whose y changed
// form L) and deep_relabel_kernel (L -> new blocks).  The bookkeeping that closes round r - 1 (block sizes, leaver
// counts, claimed slots, k) does not touch anything the front of round r reads or writes (lists and leaver counts are
// double-buffered by round parity), so it rides in the same launch as extra CTAs instead of a launch of its own.
constexpr int kDeepLaneRow = 64;  // rows up to this length are summed by the lane that found them dirty

// node i (valid on lanes with `fresh`) has a changed out-neighbour and is visited for the first time this round: new y
// under the fixed key; if it differs from the stored one the node joins L.  Every lane of the warp must call.
template <bool WEIGHTED>
__device__ __forceinline__ void
deep_visit(bool fresh, int i, const int64_t* __restrict__ row_ptr, const int* __restrict__ col,
           const u32* __restrict__ wt, const int* __restrict__ colour, u64 key, u64* __restrict__ y,
           int* __restrict__ lcount, int* __restrict__ leavers, int* __restrict__ leaver_block, u64* __restrict__ n_leavers,
           u64 ymask) {
  const int lane = threadIdx.x & 31;
  int64_t a = 0, b = 0;
  if (fresh) {
    a = row_ptr[i];
    b = row_ptr[i + 1];
  }
  const bool small = b - a <= kDeepLaneRow;
  u64 acc = 0;
  if (small) {
    for (int64_t p = a; p < b; ++p) {
      u64 v = weight_of(key, (u64)(u32)__ldcg(colour + col[p]));
      if (WEIGHTED) v *= (u64)wt[p];
      acc += v;
    }
  }
  unsigned big = __ballot_sync(0xffffffffu, !small);
  while (big) {
    const int src = __ffs(big) - 1;
    big &= big - 1;
    const int64_t ra = __shfl_sync(0xffffffffu, a, src), rb = __shfl_sync(0xffffffffu, b, src);
    u64 s = 0;
    for (int64_t p = ra + lane; p < rb; p += 32) {
      u64 v = weight_of(key, (u64)(u32)__ldcg(colour + col[p]));
      if (WEIGHTED) v *= (u64)wt[p];
      s += v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == src) acc = s;
  }
  acc &= ymask;
  const bool moved = fresh && acc != (y[i] & ymask);
  const int c = moved ? colour[i] : -1;
  const u64 pos = warp_append(moved, n_leavers);
  if (moved) {
    y[i] = acc;
    leavers[pos] = i;
    leaver_block[pos] = c;
  }
  warp_count_by_key(moved, c, lcount, +1);
}

// End of a deep round: block sizes follow the moves, leaver counts and claimed slots are reset, then the last CTA to finish
// does k += fresh ids, logs k and re-arms the counters.  `part` CTAs (indices cta .. ) share the work.
__device__ __forceinline__ void
deep_finish_part(unsigned cta, unsigned part, const int* __restrict__ leavers, const int* __restrict__ leaver_block,
                 const int* __restrict__ colour, int* __restrict__ size, int* __restrict__ lcount, Slot* __restrict__ table,
                 const u32* __restrict__ slots, u64* __restrict__ deep, int leavers_slot, int consumed_slot,
                 u64* __restrict__ scal, u64* __restrict__ log, int log_slot) {
  const u64 nl = deep[leavers_slot], ns = deep[kDeepSlots], n_new = deep[kDeepNew], k_old = scal[kScalK];
  const u64 stride = (u64)part * blockDim.x, first = (u64)cta * blockDim.x + threadIdx.x;
  for (u64 base = first - (threadIdx.x & 31); base < nl; base += stride) {  // whole-warp trips
    const u64 t = base + (threadIdx.x & 31);
    const bool valid = t < nl;
    const int c = valid ? leaver_block[t] : -1, id = valid ? colour[leavers[t]] : -1;
    const bool moved = valid && id != c;
    warp_count_by_key(moved, id, size, +1);
    warp_count_by_key(moved, c, size, -1);
    if (valid && lcount[c] != 0) lcount[c] = 0;
  }
  for (u64 t = first; t < ns; t += stride) store_slot(table + slots[t], kEmpty, kEmpty);
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const u64 ticket = atomicAdd(scal + kScalTicket, 1ull);
    if (ticket == (u64)part - 1) {  // every other finishing CTA has read the counters before taking its ticket
      scal[kScalK] = k_old + n_new;
      scal[kScalTicket] = 0;
      if (log) log[log_slot] = k_old + n_new;
      if (nl > scal[kScalFrontier]) scal[kScalFrontier] = nl;  // largest |L| since the host last looked (it picks the launch shape)
      deep[leavers_slot] = 0;
      deep[kDeepSlots] = 0;
      deep[kDeepNew] = 0;
      deep[consumed_slot] = 0;
    }
  }
}

struct DeepFinishArgs {  // the round being closed (fin_ctas == 0: nothing to close)
  unsigned fin_ctas;
  const int* leavers;
  const int* leaver_block;
  int* lcount;
  int leavers_slot, consumed_slot, log_slot;
  u64* log;
};

// CTAs [0, fin.fin_ctas) close the previous round; the others open this one: every in-neighbour of a changed node is
// visited once (mark[i] == round: already taken).  One warp takes four changed nodes per trip: in-neighbour lists of up to
// kDeepSmall entries are walked by eight lanes each (step by step, so that the appends of a step share one atomic), longer
// ones by the whole warp.  do_front == 0: only the closing part runs (end of a window).
constexpr int kDeepSmall = 64;
// the front of one round by the CTAs cta = 0 .. nctas - 1 of whatever launch runs it (a grid of its own, or a cluster)
template <bool WEIGHTED>
__device__ __forceinline__ void
deep_front_part(unsigned cta, unsigned nctas, const int* __restrict__ changed, const u64* __restrict__ n_changed,
                const int64_t* __restrict__ tp_ptr, const int* __restrict__ tp_src, int* __restrict__ mark, int round,
                const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const u32* __restrict__ wt,
                int* __restrict__ colour, u64 key, u64* __restrict__ y, int* __restrict__ lcount,
                int* __restrict__ leavers, int* __restrict__ leaver_block, u64* __restrict__ n_leavers, u64 ymask) {
  const int lane = threadIdx.x & 31, sub = lane & 7, grp = lane >> 3;
  const int64_t nc = (int64_t)*n_changed;
  // a warp takes four changed nodes per trip, eight lanes each
  const int64_t nwarps = ((int64_t)nctas * blockDim.x) >> 5;
  const int64_t warp = ((int64_t)cta * blockDim.x + threadIdx.x) >> 5;
  for (int64_t base = warp * 4; base < nc; base += nwarps * 4) {
    const int64_t t = base + grp;
    int64_t a = 0, b = 0;
    if (t < nc) {
      const int j = changed[t];
      a = tp_ptr[j];
      b = tp_ptr[j + 1];
    }
    const bool small = b - a <= kDeepSmall;
    int steps = small ? (int)((b - a + 7) >> 3) : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) steps = max(steps, __shfl_xor_sync(0xffffffffu, steps, o));
    for (int q = 0; q < steps; ++q) {
      const int64_t p = a + 8 * q + sub;
      int i = -1;
      bool fresh = false;
      if (small && p < b) {
        i = tp_src[p];
        fresh = mark[i] != round && atomicExch(mark + i, round) != round;
      }
      deep_visit<WEIGHTED>(fresh, i, row_ptr, col, wt, colour, key, y, lcount, leavers, leaver_block, n_leavers, ymask);
    }
    unsigned big = __ballot_sync(0xffffffffu, !small && sub == 0);
    while (big) {
      const int src = __ffs(big) - 1;
      big &= big - 1;
      const int64_t ra = __shfl_sync(0xffffffffu, a, src), rb = __shfl_sync(0xffffffffu, b, src);
      for (int64_t p = ra + lane; p - lane < rb; p += 32) {
        int i = -1;
        bool fresh = false;
        if (p < rb) {
          i = tp_src[p];
          fresh = mark[i] != round && atomicExch(mark + i, round) != round;
        }
        deep_visit<WEIGHTED>(fresh, i, row_ptr, col, wt, colour, key, y, lcount, leavers, leaver_block, n_leavers, ymask);
      }
    }
  }
}

template <bool WEIGHTED>
__global__ void __launch_bounds__(256)
deep_front_kernel(DeepFinishArgs fin, int do_front, const int* __restrict__ changed, const u64* __restrict__ n_changed,
                  const int64_t* __restrict__ tp_ptr, const int* __restrict__ tp_src, int* __restrict__ mark, int round,
                  const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const u32* __restrict__ wt,
                  int* __restrict__ colour, u64 key, u64* __restrict__ y, int* __restrict__ size, int* __restrict__ lcount,
                  int* __restrict__ leavers, int* __restrict__ leaver_block, u64* __restrict__ n_leavers,
                  Slot* __restrict__ table, const u32* __restrict__ slots, u64* __restrict__ deep, u64* __restrict__ scal,
                  u64 ymask) {
  if (blockIdx.x < fin.fin_ctas) {
    deep_finish_part(blockIdx.x, fin.fin_ctas, fin.leavers, fin.leaver_block, colour, size, fin.lcount, table, slots, deep,
                     fin.leavers_slot, fin.consumed_slot, scal, fin.log, fin.log_slot);
    return;
  }
  if (!do_front) return;
  deep_front_part<WEIGHTED>(blockIdx.x - fin.fin_ctas, gridDim.x - fin.fin_ctas, changed, n_changed, tp_ptr, tp_src, mark, round,
                            row_ptr, col, wt, colour, key, y, lcount, leavers, leaver_block, n_leavers, ymask);
}

// L -> new blocks.  Thread per leaver: the exact key (old colour, new y) claims or finds a slot of the relabel table; the
// claimer takes the old id if the whole block is leaving and nobody took it yet this round, otherwise a fresh id.
// Program order inside a warp is claim -> publish -> poll, so a polling lane never waits on a lane of its own warp, and a
// claimer publishes without waiting on anybody: the polls terminate.
__device__ __forceinline__ void
deep_relabel_part(unsigned cta, unsigned nctas, const int* __restrict__ leavers, const int* __restrict__ leaver_block,
                  const u64* __restrict__ n_leavers, int* __restrict__ colour, const u64* __restrict__ y,
                  const int* __restrict__ size, const int* __restrict__ lcount, int* __restrict__ inherit, int round,
                  Slot* __restrict__ table, u32 table_mask, u32* __restrict__ slots, u64* __restrict__ n_slots,
                  const u64* __restrict__ k_ptr, u64* __restrict__ n_new, int* __restrict__ changed_out,
                  u64* __restrict__ n_changed_out, u64 ymask) {
  const int64_t nl = (int64_t)*n_leavers;
  const int k_old = (int)*k_ptr;
  const int64_t stride = (int64_t)nctas * blockDim.x;
  const int64_t first = (int64_t)cta * blockDim.x + threadIdx.x;
  // whole warps iterate together (the last trip is padded) so that __syncwarp() sees every lane
  for (int64_t base = first - (threadIdx.x & 31); base < nl; base += stride) {
    const int64_t t = base + (threadIdx.x & 31);
    const bool valid = t < nl;
    bool win = false, lose = false;
    u32 slot = 0, id = kPending;
    int i = -1, c = -1;
    bool all_leave = false;
    if (valid) {
      i = leavers[t];
      c = leaver_block[t];
      const u64 yi = y[i] & ymask;
      all_leave = lcount[c] == size[c];  // issued before the probe: independent of it
      const Slot mine = {yi, (u64)(u32)c | ((u64)kPending << 32)};
      const Slot empty = {kEmpty, kEmpty};
      slot = (u32)slot_hash((u32)c, yi) & table_mask;
      while (true) {
        Slot v = load_slot(table + slot);
        if (v.y == kEmpty || v.cx == kEmpty) {
          v = cas128(table + slot, empty, mine);
          if (v.y == kEmpty && v.cx == kEmpty) {
            win = true;
            break;
          }
        }
        if (v.y == yi && (u32)v.cx == (u32)c) {
          lose = true;
          id = (u32)(v.cx >> 32);
          break;
        }
        slot = (slot + 1) & table_mask;
      }
    }
    bool fresh = false;  // a claimer that needs a new id (the block keeps its old id for somebody else)
    if (win) {
      if (all_leave && atomicExch(inherit + c, round) != round) id = (u32)c;
      else fresh = true;
    }
    const u64 fpos = warp_append(fresh, n_new);
    if (fresh) id = (u32)(k_old + (int)fpos);
    const u64 spos = warp_append(win, n_slots);
    if (win) {
      st_slot_id(table + slot, id);
      slots[spos] = slot;
    }
    __syncwarp();
    if (lose)
      while (id == kPending) id = ld_slot_id(table + slot);
    const bool moved = valid && (int)id != c;
    const u64 cpos = warp_append(moved, n_changed_out);
    if (moved) {
      colour[i] = (int)id;
      changed_out[cpos] = i;
    }
  }
}

__global__ void __launch_bounds__(256)
deep_relabel_kernel(const int* __restrict__ leavers, const int* __restrict__ leaver_block, const u64* __restrict__ n_leavers,
                    int* __restrict__ colour, const u64* __restrict__ y, const int* __restrict__ size,
                    const int* __restrict__ lcount, int* __restrict__ inherit, int round, Slot* __restrict__ table,
                    u32 table_mask, u32* __restrict__ slots, u64* __restrict__ n_slots, const u64* __restrict__ k_ptr,
                    u64* __restrict__ n_new, int* __restrict__ changed_out, u64* __restrict__ n_changed_out, u64 ymask) {
  deep_relabel_part(blockIdx.x, gridDim.x, leavers, leaver_block, n_leavers, colour, y, size, lcount, inherit, round, table,
                    table_mask, slots, n_slots, k_ptr, n_new, changed_out, n_changed_out, ymask);
}

// ---- a window of rounds in ONE launch by one thread-block cluster ------------------------------------------------------------
// A round of this regime is two launches of a few microseconds each.  A cluster of kDeepClusterCtas CTAs runs the same three parts
// (front, relabel, closing) for `rounds` rounds back to back; the phases are separated by the hardware cluster barrier
// (arrive.release / wait.acquire: a few hundred cycles, and it makes the other CTAs' global writes visible) instead of kernel
// boundaries.  Same device functions, same data, same results as the two-kernel form.  Measured on B200 and NOT the default
// (WL_FLAG_DEEP_CLUSTER): what bounds a round is its two dependent chains of about ten L2 accesses, not the launches, and eight
// SMs are too few for the 26 k leavers per round of the 2048^2 grid (profiles/r2b_deep_cluster.md).
constexpr int kDeepClusterCtas = 8;      // portable cluster size
constexpr int kDeepClusterThreads = 1024;
struct DeepClusterArgs {
  int* changed[2];
  int* lcount[2];
  int* leavers[2];
  int* leaver_block[2];
  const int64_t* tp_ptr;
  const int* tp_src;
  int* mark;
  const int64_t* row_ptr;
  const int* col;
  const u32* wt;
  int* colour;
  u64 key;
  u64* y;
  int* size;
  int* inherit;
  Slot* table;
  u32 table_mask;
  u32* slots;
  u64* deep;
  u64* scal;
  u64 ymask;
  int round0, rounds;
};
__device__ __forceinline__ void cluster_barrier() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
template <bool WEIGHTED>
__global__ void __launch_bounds__(kDeepClusterThreads, 1)
deep_cluster_kernel(const DeepClusterArgs a) {
  const unsigned cta = blockIdx.x, nctas = gridDim.x;  // the grid is one cluster
  for (int j = 0; j < a.rounds; ++j) {
    const int round = a.round0 + j, in = round & 1, out = in ^ 1;
    if (j > 0)  // close round - 1 (touches nothing the front of this round reads or writes, see deep_front_kernel)
      deep_finish_part(cta, nctas, a.leavers[out], a.leaver_block[out], a.colour, a.size, a.lcount[out], a.table, a.slots, a.deep,
                       kDeepLeavers0 + out, kDeepChanged0 + out, a.scal, a.scal + kScalLog, j - 1);
    deep_front_part<WEIGHTED>(cta, nctas, a.changed[in], a.deep + kDeepChanged0 + in, a.tp_ptr, a.tp_src, a.mark, round, a.row_ptr,
                              a.col, a.wt, a.colour, a.key, a.y, a.lcount[in], a.leavers[in], a.leaver_block[in],
                              a.deep + kDeepLeavers0 + in, a.ymask);
    cluster_barrier();
    deep_relabel_part(cta, nctas, a.leavers[in], a.leaver_block[in], a.deep + kDeepLeavers0 + in, a.colour, a.y, a.size,
                      a.lcount[in], a.inherit, round, a.table, a.table_mask, a.slots, a.deep + kDeepSlots, a.scal + kScalK,
                      a.deep + kDeepNew, a.changed[out], a.deep + kDeepChanged0 + out, a.ymask);
    cluster_barrier();
  }
  const int last = (a.round0 + a.rounds - 1) & 1;
  deep_finish_part(cta, nctas, a.leavers[last], a.leaver_block[last], a.colour, a.size, a.lcount[last], a.table, a.slots, a.deep,
                   kDeepLeavers0 + last, kDeepChanged0 + last, a.scal, a.scal + kScalLog, a.rounds - 1);
}

}  // namespace wl
