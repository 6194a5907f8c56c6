// =====================================================================================
// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product.
//
// Plain, slow, obviously-correct CPU implementations of what the CUDA path computes,
// written from /root/reference/PAPER.md (arxiv/paper_2607_02603).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// this file.  It shares no code, header, table or constant generator with
// paper_2607_02603_b200/csrc (the CUDA path); neither side includes the other.
//
// What is here, each with the passage it follows:
//   oracle_refine        coarsest stable colouring refining an initial partition
//                        (Def. 1-3; L94) by classical signature-sort refinement
//                        (deterministic, no hashing, no randomness).      PINNED (tests/test_oracle_pins.py:
//                        brute force <= 7 nodes, closed forms, renumbering invariance)
//   oracle_is_stable     Def. 1 (L47-L49) checked literally per node against its block's first node.   PINNED
//                        (against a dense numpy A.S product in tests)
//   oracle_canonical     first-occurrence renumbering of a colour vector.                 PINNED (hand cases)
//   oracle_inner_labels  Def. 5 (L139-L145) via per-node batch labels (L463).             PINNED (set brute force)
//   oracle_quotient      Def. 4 / Eq. 1 (L59-L65), representative = minimum node index.   PINNED (dense A.S = S.A')
//   oracle_rbsc          Algorithm 2 (L169-L202) with oracle_refine in place of RSC.     PINNED (Thm 2 invariants,
//                        N_b = 1 equality, order independence; the L328 stop rule: equals the plain loop cut after the
//                        iteration a Python restatement of the rule names)
//   oracle_rbsc_init     the same from initial classes (reading Q18: Eq. 3 intersected with them). PINNED (stable, refines
//                        the classes and oracle_refine(init), equals it on one batch, naming independence, hand cases)
//   oracle_weight        the keyed bijection w = P_key(colour) that DESIGN.md §"Readings" Q4/Q5 fixes in place of
//                        the paper's unseeded xoshiro/SplitMix recipe (L467-L473).  Bit stream: PARITY UNPINNED
//                        (the paper prints no test vectors); bijectivity and constants are pinned.
//   oracle_spmv_u64      z = A w mod 2^64 (Alg. 1 line 5, L120), serial.                  PINNED (numpy uint64 dense product)
//   oracle_rsc           Algorithm 1 (L106-L127) step by step in Z/2^64 with oracle_weight. PINNED (equals oracle_refine,
//                        reduced-q miss rate 2^{t-q} of Lemma 1)
//
// Conventions: CSR rows are sources (out-edges, L43/L49).  row_ptr int64[n+1], col int32[m],
// wt uint32[m] or NULL (all ones).  Duplicate (i,j) entries add (a_ij in N_0, L43).
// =====================================================================================
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <map>
#include <utility>
#include <vector>

typedef int64_t i64;
typedef int32_t i32;
typedef uint64_t u64;
typedef uint32_t u32;

namespace {

// first-occurrence renumbering: ids 0,1,2,... in order of the first node carrying each label
i64 canonical(i64 n, const i32* in, i32* out) {
  std::map<i32, i32> seen;
  for (i64 i = 0; i < n; ++i) {
    auto it = seen.find(in[i]);
    if (it == seen.end()) {
      i32 id = (i32)seen.size();
      seen.emplace(in[i], id);
      out[i] = id;
    } else {
      out[i] = it->second;
    }
  }
  return (i64)seen.size();
}

// signature of node i under colouring c: sorted list of (colour of out-neighbour, summed weight)
typedef std::vector<std::pair<i32, u64>> Sig;

void build_sig(i64 i, const i64* row_ptr, const i32* col, const u32* wt, const i32* c, Sig& s) {
  s.clear();
  for (i64 e = row_ptr[i]; e < row_ptr[i + 1]; ++e) s.emplace_back(c[col[e]], wt ? (u64)wt[e] : 1ull);
  std::sort(s.begin(), s.end());
  // merge equal colours: a_{i,B'} = sum_{l in B'} a_il  (Def. 1)
  size_t o = 0;
  for (size_t k = 0; k < s.size();) {
    i32 colr = s[k].first;
    u64 sum = 0;
    while (k < s.size() && s[k].first == colr) sum += s[k++].second;
    if (sum != 0) s[o++] = std::make_pair(colr, sum);
  }
  s.resize(o);
}

}  // namespace

extern "C" {

i64 oracle_canonical(i64 n, const i32* in, i32* out) { return canonical(n, in, out); }

// ---------------------------------------------------------------------------------
// Def. 1 (L47-L49): for every block B, B' and i, j in B: sum_{l in B'} a_il == sum_{l in B'} a_jl.
// Checked by comparing every node's merged signature with that of the first node of its block.
// returns 1 stable, 0 not.
// ---------------------------------------------------------------------------------
int oracle_is_stable(i64 n, const i64* row_ptr, const i32* col, const u32* wt, const i32* colors) {
  std::map<i32, Sig> first_sig;
  Sig s;
  for (i64 i = 0; i < n; ++i) {
    build_sig(i, row_ptr, col, wt, colors, s);
    auto it = first_sig.find(colors[i]);
    if (it == first_sig.end())
      first_sig.emplace(colors[i], s);
    else if (it->second != s)
      return 0;
  }
  return 1;
}

// ---------------------------------------------------------------------------------
// Coarsest stable colouring refining `init` (NULL = one block), L94 / Def. 3.
// Round: signature(i) = (c(i), merged sorted neighbour-colour list); sort nodes by signature;
// dense ids in sorted order; stop when the number of ids equals the previous round's
// (a refinement with the same block count is the same partition, L153).
// counts[r] = number of colours after round r+1 (r < max_rounds); *rounds = rounds executed
// (the last one only confirms).  out = canonical first-occurrence ids.  returns final count, or -1
// if max_rounds was hit before convergence.
// ---------------------------------------------------------------------------------
i64 oracle_refine(i64 n, const i64* row_ptr, const i32* col, const u32* wt, const i32* init, i32* out,
                  i32 max_rounds, i64* counts, i32* rounds) {
  std::vector<i32> c(n), nc(n);
  i64 k;
  if (init) {
    k = canonical(n, init, c.data());
  } else {
    std::fill(c.begin(), c.end(), 0);
    k = n > 0 ? 1 : 0;
  }
  *rounds = 0;
  if (n == 0) return 0;
  std::vector<Sig> sig(n);
  std::vector<i64> order(n);
  for (i32 r = 0; r < max_rounds; ++r) {
#pragma omp parallel for schedule(dynamic, 1024)
    for (i64 i = 0; i < n; ++i) build_sig(i, row_ptr, col, wt, c.data(), sig[i]);
    for (i64 i = 0; i < n; ++i) order[i] = i;
    auto less = [&](i64 a, i64 b) {
      if (c[a] != c[b]) return c[a] < c[b];
      return sig[a] < sig[b];  // lexicographic on (colour, weight) lists
    };
    std::sort(order.begin(), order.end(), less);
    i64 knew = 0;
    for (i64 p = 0; p < n; ++p) {
      if (p > 0 && (less(order[p - 1], order[p]) || less(order[p], order[p - 1]))) ++knew;
      nc[order[p]] = (i32)knew;
    }
    ++knew;
    c.swap(nc);
    if (counts) counts[r] = knew;
    *rounds = r + 1;
    if (knew == k) {
      canonical(n, c.data(), out);
      return knew;
    }
    k = knew;
  }
  canonical(n, c.data(), out);
  return -1;
}

// ---------------------------------------------------------------------------------
// Def. 5 (L139-L145) with the method of L463: every edge adds its batch label to its source; a node
// whose labels are all equal to k is inner to batch k; several distinct labels -> boundary (-1).
// A node with no out-edge is vacuously inner to every batch (L141); reading Q9 assigns it to
// `sink_batch[i]` (given by the caller).  edge_batch[e] = batch of CSR edge slot e.
// ---------------------------------------------------------------------------------
void oracle_inner_labels(i64 n, const i64* row_ptr, const i32* edge_batch, const i32* sink_batch, i32* label) {
  for (i64 i = 0; i < n; ++i) {
    if (row_ptr[i] == row_ptr[i + 1]) {
      label[i] = sink_batch[i];
      continue;
    }
    i32 b = edge_batch[row_ptr[i]];
    bool inner = true;
    for (i64 e = row_ptr[i]; e < row_ptr[i + 1]; ++e)
      if (edge_batch[e] != b) inner = false;
    label[i] = inner ? b : -1;
  }
}

// ---------------------------------------------------------------------------------
// Def. 4 / Eq. 1 (L59-L65): quotient (H, A') of a stable colouring given as canonical colours
// (ids 0..k-1 by first occurrence, so the first node of a block is its minimum index = representative).
// a'_{B,B'} = sum_{l in B'} a_{i_B,l}.  Output CSR with sorted columns, zero entries dropped.
// q_row_ptr int64[k+1]; q_col/q_wt sized >= m (upper bound).  returns number of entries.
// ---------------------------------------------------------------------------------
i64 oracle_quotient(i64 n, const i64* row_ptr, const i32* col, const u32* wt, const i32* colors, i64 k,
                    i64* q_row_ptr, i32* q_col, u32* q_wt) {
  std::vector<i64> rep(k, -1);
  for (i64 i = 0; i < n; ++i)
    if (rep[colors[i]] < 0) rep[colors[i]] = i;
  Sig s;
  i64 out = 0;
  q_row_ptr[0] = 0;
  for (i64 b = 0; b < k; ++b) {
    build_sig(rep[b], row_ptr, col, wt, colors, s);
    for (auto& p : s) {
      q_col[out] = p.first;
      q_wt[out] = (u32)p.second;
      ++out;
    }
    q_row_ptr[b + 1] = out;
  }
  return out;
}

// ---------------------------------------------------------------------------------
// Algorithm 2 (L169-L202) with oracle_refine in place of RSC, for the library's default edge
// partition (readings Q13-Q17): batches = consecutive runs of the CSR edge array cut by
// `first_cuts` in outer iteration 1 (ncuts+1 entries) and by the same greedy row-boundary rule with
// cap max_batch_edges afterwards.  Arbitrary first partitions: first_edge_batch != NULL (batch id per
// edge slot, nb0 batches).  out = colours on the ORIGINAL nodes (canonical).  Returns final colour count.
// stats[0] = outer iterations, stats[1] = N_b of the last iteration.
// ---------------------------------------------------------------------------------
static void greedy_cuts(i64 n, const i64* rp, i64 cap, std::vector<i64>& cuts) {
  i64 m = rp[n];
  cuts.assign(1, 0);
  while (cuts.back() < m) {
    i64 start = cuts.back(), limit = start + cap;
    if (limit >= m) {
      cuts.push_back(m);
      break;
    }
    // largest row boundary <= limit that is > start, else split inside the row
    i64 best = -1;
    for (i64 r = 0; r <= n; ++r)
      if (rp[r] <= limit && rp[r] > start) best = rp[r];
    cuts.push_back(best > 0 ? best : limit);
  }
}

// inherit != 0 (reading Q14b): from the second outer iteration on the edge partition is not re-cut by M_b;
// the quotient inherits the batches of its graph: batch k of the quotient = the blocks whose representative row is complete
// once batch k of the graph has been read (in node order), with exactly their rows.  L163 allows any partition.
// aggressive != 0 (L328, the termination used for Table 4): "the outer loop of Algorithm 2 stops as soon as the number of
// batches in the next iteration would not decrease": after the quotient of an iteration that ran with N_b batches has been
// built, the edge partition of the next iteration is made as usual; if it has >= N_b batches the loop ends with the
// colouring reached so far (every outer iteration ends on a stable colouring, Thm 2 / L206).
// init0 != NULL (reading Q18; optional extension): Algorithm 2 has no initial partition (L171), Algorithm 1
// has (L94).  With init classes the local start of batch k is Eq. 3's partition intersected with them: the inner nodes of batch k
// are grouped by their class, every other node stays a singleton (L151).  A node of a quotient graph (a block, Def. 4) carries the
// class of its nodes: every H_k refines its start, so a block never spans two classes.  Everything else is Algorithm 2 as written.
i64 oracle_rbsc_init(i64 n0, const i64* row_ptr0, const i32* col0, const u32* wt0, const i32* init0, i64 max_batch_edges,
                     i32 nb0, const i64* first_cuts, const i32* first_edge_batch, i32 max_outer, i32 inherit, i32 aggressive,
                     i32* out, i64* stats) {
  i64 n = n0;
  std::vector<i32> cls(n0, 0);  // class of every node of the current graph, dense ids (first occurrence)
  if (init0) canonical(n0, init0, cls.data());
  std::vector<i64> rp(row_ptr0, row_ptr0 + n0 + 1);
  std::vector<i32> col(col0, col0 + rp[n0]);
  std::vector<u32> wt(rp[n0]);
  for (i64 e = 0; e < rp[n0]; ++e) wt[e] = wt0 ? wt0[e] : 1u;
  std::vector<i32> map(n0);  // original node -> current node
  for (i64 i = 0; i < n0; ++i) map[i] = (i32)i;
  i32 outer = 0;
  i64 nb_last = 0;
  std::vector<i64> inh_cuts, inh_nodes;  // inherit: edge cuts and node ranges of the coming iteration
  while (true) {
    ++outer;
    i64 m = rp[n];
    std::vector<i32> eb(m);
    i64 nb;
    std::vector<i64> cuts, node_cuts;
    if (inherit && outer > 1) {
      cuts = inh_cuts;
      node_cuts = inh_nodes;
      nb = (i64)cuts.size() - 1;
      for (i64 k = 0; k < nb; ++k)
        for (i64 e = cuts[k]; e < cuts[k + 1]; ++e) eb[e] = (i32)k;
    } else if (outer == 1 && first_edge_batch) {
      nb = nb0;
      for (i64 e = 0; e < m; ++e) eb[e] = first_edge_batch[e];
    } else {
      if (outer == 1 && first_cuts)
        cuts.assign(first_cuts, first_cuts + nb0 + 1);
      else
        greedy_cuts(n, rp.data(), max_batch_edges, cuts);
      nb = (i64)cuts.size() - 1;
      if (nb < 1) nb = 1;  // m == 0: one empty batch
      for (i64 k = 0; k + 1 < (i64)cuts.size(); ++k)
        for (i64 e = cuts[k]; e < cuts[k + 1]; ++e) eb[e] = (i32)k;
    }
    // sinks: batch whose edge range contains the row's (empty) position; batch 0 for arbitrary partitions (Q9)
    std::vector<i32> sink(n, 0);
    if (!node_cuts.empty()) {  // inherited batches come with their node ranges
      for (i64 k = 0; k < nb; ++k)
        for (i64 i = node_cuts[k]; i < node_cuts[k + 1]; ++i) sink[i] = (i32)k;
    } else if (!cuts.empty())
      for (i64 i = 0; i < n; ++i)
        if (rp[i] == rp[i + 1]) {
          i64 k = 0;
          while (k + 1 < nb && cuts[k + 1] <= rp[i]) ++k;
          sink[i] = (i32)k;
        }
    std::vector<i32> label(n);
    oracle_inner_labels(n, rp.data(), eb.data(), sink.data(), label.data());
    // Alg. 2 lines 7-13: per batch local refinement from H_k^0 (Eq. 3), then merge (Eq. 4)
    std::vector<i32> H(n, -1);
    i64 next_id = 0;
    for (i64 k = 0; k < nb; ++k) {
      // A|E_k as a CSR over all n nodes
      std::vector<i64> brp(n + 1, 0);
      std::vector<i32> bcol;
      std::vector<u32> bwt;
      for (i64 i = 0; i < n; ++i) {
        for (i64 e = rp[i]; e < rp[i + 1]; ++e)
          if (eb[e] == k) {
            bcol.push_back(col[e]);
            bwt.push_back(wt[e]);
          }
        brp[i + 1] = (i64)bcol.size();
      }
      // H_k^0: inner nodes of k share one block, everyone else is a singleton (Eq. 3)
      // (with init classes, Q18: inner nodes keep their class id c < n, node i outside V_k is the singleton n + i)
      std::vector<i32> init(n), loc(n);
      for (i64 i = 0; i < n; ++i) init[i] = (label[i] == k) ? cls[i] : (i32)(n + i);
      i32 rounds;
      i64 kk = oracle_refine(n, brp.data(), bcol.data(), bwt.data(), init.data(), loc.data(), (i32)(n + 2), nullptr, &rounds);
      (void)kk;
      // collect blocks that lie inside V_k (Eq. 4): since H_k refines H_k^0, those are the blocks of inner nodes
      std::map<i32, i32> ids;
      for (i64 i = 0; i < n; ++i)
        if (label[i] == k) {
          auto it = ids.find(loc[i]);
          if (it == ids.end()) it = ids.emplace(loc[i], (i32)(next_id++)).first;
          H[i] = it->second;
        }
    }
    for (i64 i = 0; i < n; ++i)
      if (H[i] < 0) H[i] = (i32)(next_id++);  // boundary singletons (Alg. 2 l.11-12)
    std::vector<i32> Hc(n);
    i64 k = canonical(n, H.data(), Hc.data());
    // quotient (Alg. 2 l.13)
    std::vector<i64> qrp(k + 1);
    std::vector<i32> qcol(m > 0 ? m : 1);
    std::vector<u32> qwt(m > 0 ? m : 1);
    i64 qm = oracle_quotient(n, rp.data(), col.data(), wt.data(), Hc.data(), k, qrp.data(), qcol.data(), qwt.data());
    for (i64 i = 0; i < n0; ++i) map[i] = Hc[map[i]];
    {  // class of a block = class of its first node (canonical ids are numbered by first node)
      std::vector<i32> next_cls;
      for (i64 i = 0; i < n; ++i)
        if ((i64)Hc[i] == (i64)next_cls.size()) next_cls.push_back(cls[i]);
      cls.swap(next_cls);
    }
    if (inherit && !cuts.empty()) {
      // batch j of the quotient: blocks whose first node lies before done_nodes(j) = the nodes whose row is complete after
      // batch j (all nodes after the last batch), minus the blocks of earlier batches; batches without blocks disappear
      inh_cuts.assign(1, 0);
      inh_nodes.assign(1, 0);
      for (i64 j = 0; j < nb; ++j) {
        i64 done_nodes;
        if (!node_cuts.empty()) done_nodes = node_cuts[j + 1];
        else if (j == nb - 1) done_nodes = n;
        else {
          done_nodes = 0;
          while (done_nodes < n && rp[done_nodes + 1] <= cuts[j + 1]) ++done_nodes;
        }
        i64 done_blocks = 0;  // canonical ids are ordered by first node: blocks with first node < done_nodes
        for (i64 i = 0; i < done_nodes; ++i) done_blocks = std::max<i64>(done_blocks, (i64)Hc[i] + 1);
        if (done_blocks > inh_nodes.back()) {
          inh_nodes.push_back(done_blocks);
          inh_cuts.push_back(qrp[done_blocks]);
        }
      }
    }
    bool stop = (nb == 1) || (k == n);  // Alg. 2 l.15 (L200), reading Q15
    nb_last = nb;
    rp.assign(qrp.begin(), qrp.end());
    col.assign(qcol.begin(), qcol.begin() + qm);
    wt.assign(qwt.begin(), qwt.begin() + qm);
    n = k;
    if (stop || outer >= max_outer) break;
    if (aggressive) {  // L328: N_b of the next iteration
      i64 nb_next;
      if (inherit && !inh_cuts.empty()) {
        nb_next = (i64)inh_cuts.size() - 1;
      } else {
        std::vector<i64> next_cuts;
        greedy_cuts(n, rp.data(), max_batch_edges, next_cuts);
        nb_next = (i64)next_cuts.size() - 1;
      }
      if (nb_next < 1) nb_next = 1;
      if (nb_next >= nb) break;
    }
  }
  if (stats) {
    stats[0] = outer;
    stats[1] = nb_last;
  }
  return canonical(n0, map.data(), out);
}

i64 oracle_rbsc(i64 n0, const i64* row_ptr0, const i32* col0, const u32* wt0, i64 max_batch_edges,
                i32 nb0, const i64* first_cuts, const i32* first_edge_batch, i32 max_outer, i32 inherit, i32 aggressive,
                i32* out, i64* stats) {
  return oracle_rbsc_init(n0, row_ptr0, col0, wt0, nullptr, max_batch_edges, nb0, first_cuts, first_edge_batch, max_outer, inherit,
                          aggressive, out, stats);
}

// ---------------------------------------------------------------------------------
// Weight function (readings Q4/Q5; replaces L467-L473's unseeded recipe):
//   mix(x):  x ^= x >> 32;  x *= M1;  x ^= x >> 29;  x *= M2;  x ^= x >> 32      (all mod 2^64)
//   M1 = floor(frac(sqrt 2) 2^64) | 1,  M2 = floor(frac(sqrt 3) 2^64) | 1,  G = floor(frac(golden ratio) 2^64) | 1
//   key(seed, stream, round) = mix( mix( mix(seed + G) + stream ) + round )
//   w(c) = mix(c + key)                c = dense colour id  (< 2^32)
// mix is a bijection of Z/2^64 (odd multipliers, xor-shifts), so weights of distinct colours are distinct
// (Alg. 1 lines 3-4, L115-L118, hold by construction).
// ---------------------------------------------------------------------------------
static inline u64 omix(u64 x) {
  x ^= x >> 32;
  x *= 0x6a09e667f3bcc909ull;
  x ^= x >> 29;
  x *= 0xbb67ae8584caa73bull;
  x ^= x >> 32;
  return x;
}
u64 oracle_round_key(u64 seed, u64 stream, u64 round) {
  return omix(omix(omix(seed + 0x9e3779b97f4a7c15ull) + stream) + round);
}
u64 oracle_weight(u64 key, u64 c) { return omix(c + key); }

// z = A w mod 2^q (Alg. 1 line 5, L120).  w is per NODE here (already symmetric on H).  qbits in [1,64].
void oracle_spmv_u64(i64 n, const i64* row_ptr, const i32* col, const u32* wt, const u64* w, i32 qbits, u64* z) {
  u64 mask = qbits >= 64 ? ~0ull : ((1ull << qbits) - 1);
  for (i64 i = 0; i < n; ++i) {
    u64 acc = 0;
    for (i64 e = row_ptr[i]; e < row_ptr[i + 1]; ++e) acc += (wt ? (u64)wt[e] : 1ull) * w[col[e]];
    z[i] = acc & mask;
  }
}

// ---------------------------------------------------------------------------------
// Algorithm 1 (L106-L127), reading Q1/Q2: keep the previous partition, refine, stop when the block
// count is unchanged.  Per round r (1-based): key = oracle_round_key(seed, stream, r); w_i = weight(key, c_i)
// masked to q bits; z = A w mod 2^q; new partition = dense ids of the lexicographically sorted pairs (c_i, z_i)
// (L92, L122).  z_out (may be NULL) receives z of round `z_round`.  Same outputs as oracle_refine.
// With qbits < 64 weights of distinct colours may coincide; the pair key still contains the old colour, so the
// result remains a refinement (used only by the Lemma 1 miss-rate pin).
// ---------------------------------------------------------------------------------
i64 oracle_rsc(i64 n, const i64* row_ptr, const i32* col, const u32* wt, const i32* init, u64 seed, u64 stream,
               i32 qbits, i32* out, i32 max_rounds, i64* counts, i32* rounds, i32 z_round, u64* z_out) {
  std::vector<i32> c(n), nc(n);
  i64 k;
  if (init) {
    k = canonical(n, init, c.data());
  } else {
    std::fill(c.begin(), c.end(), 0);
    k = n > 0 ? 1 : 0;
  }
  *rounds = 0;
  if (n == 0) return 0;
  u64 mask = qbits >= 64 ? ~0ull : ((1ull << qbits) - 1);
  std::vector<u64> w(n), z(n);
  std::vector<i64> order(n);
  for (i32 r = 1; r <= max_rounds; ++r) {
    u64 key = oracle_round_key(seed, stream, (u64)r);
    for (i64 i = 0; i < n; ++i) w[i] = oracle_weight(key, (u64)c[i]) & mask;
    oracle_spmv_u64(n, row_ptr, col, wt, w.data(), qbits, z.data());
    if (z_out && r == z_round) std::memcpy(z_out, z.data(), sizeof(u64) * n);
    for (i64 i = 0; i < n; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](i64 a, i64 b) {
      if (c[a] != c[b]) return c[a] < c[b];
      return z[a] < z[b];
    });
    i64 knew = 0;
    for (i64 p = 0; p < n; ++p) {
      if (p > 0 && (c[order[p]] != c[order[p - 1]] || z[order[p]] != z[order[p - 1]])) ++knew;
      nc[order[p]] = (i32)knew;
    }
    ++knew;
    c.swap(nc);
    if (counts) counts[r - 1] = knew;
    *rounds = r;
    if (knew == k) {
      canonical(n, c.data(), out);
      return knew;
    }
    k = knew;
  }
  canonical(n, c.data(), out);
  return -1;
}

}  // extern "C"
