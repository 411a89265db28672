// Length-bucketing batch scheduler (host only).  PAPER.md:113: sort the proteins by length so that one compiled
// model serves all of them; here one binary serves every shape, and bucketing bounds the padding waste while
// batching amortises launch overhead on small buckets.
#include "../../include/pf_evoformer.h"

#include <algorithm>
#include <new>
#include <vector>

struct pf_sched {
  std::vector<int> buckets;
  size_t budget;
  int S;
  struct Item { int id, len, bucket; };
  std::vector<Item> items;
  bool frozen = false;
  size_t cursor = 0;
};

extern "C" size_t pf_sched_bytes_per_protein(int bucket, int S) {
  // fp32 residual streams + bf16 workspace of the PF_BF16 path (see arena_layout in pf_api.cu):
  // msa S*N*256*(4 + 2*(1+4+1+1)) + pair N*N*128*(4 + 2*(1+1+1+1+1) + 4) bytes, rounded up generously.
  size_t N = (size_t)bucket, s = (size_t)S;
  return s * N * 256 * 18 + N * N * 128 * 20 + N * N * 8 * 2;
}

extern "C" pf_status pf_sched_create(pf_sched_t** out, const int* buckets, int n_buckets, size_t mem_budget_bytes, int S) {
  if (!out || !buckets || n_buckets < 1 || S < 1) return PF_ERR_INVALID_ARG;
  for (int i = 0; i < n_buckets; ++i)
    if (buckets[i] < 1 || (i && buckets[i] <= buckets[i - 1])) return PF_ERR_INVALID_ARG;
  pf_sched* s = new (std::nothrow) pf_sched();
  if (!s) return PF_ERR_ALLOC;
  s->buckets.assign(buckets, buckets + n_buckets);
  s->budget = mem_budget_bytes;
  s->S = S;
  *out = s;
  return PF_OK;
}

extern "C" pf_status pf_sched_add(pf_sched_t* s, int protein_id, int length) {
  if (!s) return PF_ERR_INVALID_ARG;
  if (s->frozen) return PF_ERR_INVALID_ARG;
  if (length < 1 || length > s->buckets.back()) return PF_ERR_SHAPE;
  int bucket = *std::lower_bound(s->buckets.begin(), s->buckets.end(), length);
  s->items.push_back({protein_id, length, bucket});
  return PF_OK;
}

extern "C" int pf_sched_next_batch(pf_sched_t* s, int* ids_out, int* lengths_out, int cap, int* bucket_out) {
  if (!s || !ids_out || !bucket_out || cap < 1) return -1;
  if (!s->frozen) {
    // largest first (the paper compiles for the largest protein first); stable for equal lengths
    std::stable_sort(s->items.begin(), s->items.end(),
                     [](const pf_sched::Item& a, const pf_sched::Item& b) { return a.len > b.len; });
    s->frozen = true;
  }
  if (s->cursor >= s->items.size()) return 0;
  int bucket = s->items[s->cursor].bucket;
  size_t per = pf_sched_bytes_per_protein(bucket, s->S);
  size_t maxb = per ? s->budget / per : 1;
  if (maxb < 1) maxb = 1;
  if (maxb > (size_t)cap) maxb = (size_t)cap;
  int n = 0;
  while (s->cursor < s->items.size() && (size_t)n < maxb && s->items[s->cursor].bucket == bucket) {
    ids_out[n] = s->items[s->cursor].id;
    if (lengths_out) lengths_out[n] = s->items[s->cursor].len;
    ++n;
    ++s->cursor;
  }
  *bucket_out = bucket;
  return n;
}

// Per-protein cost model for list sharding: GEMM FLOPs of one Evoformer block at the protein's bucket (SURVEY.md §8(d)
// F(S, N) with the AlphaFold dims); only ratios matter.
extern "C" double pf_sched_cost(int bucket, int S) {
  const double N = bucket, s = S, cm = 256, cz = 128, co = 32, hm = 8, hz = 4;
  return 36 * s * N * cm * cm + 4 * s * N * N * cm + 4 * N * s * s * cm + 4 * s * N * cm * co + 2 * s * N * N * co * co +
         2 * N * N * co * co * cz + 60 * N * N * cz * cz + 12 * N * N * N * cz + 2 * N * N * cz * hm + 4 * N * N * cz * hz;
}

// Replicas-only multi-GPU (independent single-GPU tasks, no communication): assign every
// protein to one of `world` ranks, longest-processing-time first over pf_sched_cost of its bucket, ties to the lowest rank.
extern "C" pf_status pf_sched_partition(const int* lengths, int n, const int* buckets, int n_buckets, int S, int world,
                                        int* rank_out) {
  if (!lengths || !buckets || !rank_out || n < 0 || n_buckets < 1 || S < 1 || world < 1) return PF_ERR_INVALID_ARG;
  for (int i = 0; i < n_buckets; ++i)
    if (buckets[i] < 1 || (i && buckets[i] <= buckets[i - 1])) return PF_ERR_INVALID_ARG;
  std::vector<int> order(n);
  std::vector<double> cost(n);
  for (int i = 0; i < n; ++i) {
    if (lengths[i] < 1 || lengths[i] > buckets[n_buckets - 1]) return PF_ERR_SHAPE;
    order[i] = i;
    cost[i] = pf_sched_cost(*std::lower_bound(buckets, buckets + n_buckets, lengths[i]), S);
  }
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost[a] > cost[b]; });
  std::vector<double> load(world, 0.0);
  for (int i : order) {
    int r = (int)(std::min_element(load.begin(), load.end()) - load.begin());
    rank_out[i] = r;
    load[r] += cost[i];
  }
  return PF_OK;
}

extern "C" void pf_sched_destroy(pf_sched_t* s) { delete s; }
