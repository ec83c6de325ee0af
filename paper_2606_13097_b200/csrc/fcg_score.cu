// Locality score of the cache management scheme (Eq. 3, 8, 9, 10): host-only bookkeeping
// that tells the caller which function entries to keep on the GPU and which to hand to fcg_segment_offload.
// No CUDA here; compiled into libfcg.so with the rest.  Readings: DESIGN.md R24.
#include <stdint.h>

#include <algorithm>
#include <map>
#include <set>
#include <utility>
#include <vector>

#include "../../include/fcg.h"

struct fcg_scorer {
  std::map<int32_t, int64_t> count;                        // invocations per function
  std::map<std::pair<int32_t, int32_t>, int64_t> follow;   // (k, j): times j was the next invocation after k
  std::map<int32_t, double> ppl;
  std::set<int32_t> last;                                  // functions of the most recent trace (l_curr = 1)

  double score(int32_t f, double alpha, double beta, double gamma) const {
    if (last.count(f)) return 1.0;
    int64_t max_cnt = 0;
    for (auto &kv : count) max_cnt = std::max(max_cnt, kv.second);
    auto it = count.find(f);
    const int64_t cnt = it == count.end() ? 0 : it->second;
    const double freq = max_cnt ? (double)cnt / (double)max_cnt : 0.0;                  // Eq. 8
    int64_t next_total = 0;
    for (auto fit = follow.lower_bound({f, INT32_MIN}); fit != follow.end() && fit->first.first == f; ++fit)
      next_total += fit->second;
    const double asso = cnt ? (double)next_total / (double)cnt : 0.0;                   // sum_j of Eq. 9
    double max_ppl = 0.0;
    for (auto &kv : ppl) max_ppl = std::max(max_ppl, kv.second);
    auto pit = ppl.find(f);
    const double sema = (max_ppl > 0.0 && pit != ppl.end()) ? pit->second / max_ppl : 0.0;   // Eq. 10
    return alpha * freq + beta * asso + gamma * sema;                                   // Eq. 3 with l_curr = 0
  }
};

extern "C" {

fcg_status_t fcg_scorer_create(fcg_scorer_t **out) {
  if (!out) return FCG_ERR_INVALID_ARG;
  *out = new fcg_scorer();
  return FCG_OK;
}

fcg_status_t fcg_scorer_destroy(fcg_scorer_t *s) {
  if (!s) return FCG_ERR_INVALID_ARG;
  delete s;
  return FCG_OK;
}

fcg_status_t fcg_scorer_record(fcg_scorer_t *s, const int32_t *ids, int32_t n) {
  if (!s || n < 0 || (n > 0 && !ids)) return FCG_ERR_INVALID_ARG;
  for (int32_t i = 0; i < n; ++i) s->count[ids[i]]++;
  for (int32_t i = 0; i + 1 < n; ++i)
    if (ids[i] != ids[i + 1]) s->follow[{ids[i], ids[i + 1]}]++;
  s->last.clear();
  s->last.insert(ids, ids + n);
  return FCG_OK;
}

fcg_status_t fcg_scorer_set_ppl(fcg_scorer_t *s, int32_t id, double ppl) {
  if (!s || !(ppl >= 0.0)) return FCG_ERR_INVALID_ARG;
  s->ppl[id] = ppl;
  return FCG_OK;
}

fcg_status_t fcg_scorer_forget(fcg_scorer_t *s, int32_t id) {
  if (!s) return FCG_ERR_INVALID_ARG;
  s->count.erase(id);
  s->ppl.erase(id);
  s->last.erase(id);
  for (auto it = s->follow.begin(); it != s->follow.end();)
    it = (it->first.first == id || it->first.second == id) ? s->follow.erase(it) : std::next(it);
  return FCG_OK;
}

fcg_status_t fcg_scorer_score(fcg_scorer_t *s, int32_t id, double alpha, double beta, double gamma, double *score) {
  if (!s || !score) return FCG_ERR_INVALID_ARG;
  *score = s->score(id, alpha, beta, gamma);
  return FCG_OK;
}

fcg_status_t fcg_scorer_rank(fcg_scorer_t *s, const int32_t *ids, int32_t n, double alpha, double beta, double gamma,
                             int32_t *ids_out, double *scores_out) {
  if (!s || n < 0 || (n > 0 && (!ids || !ids_out))) return FCG_ERR_INVALID_ARG;
  std::vector<std::pair<double, int32_t>> v;
  v.reserve(n);
  for (int32_t i = 0; i < n; ++i) v.push_back({s->score(ids[i], alpha, beta, gamma), ids[i]});
  std::sort(v.begin(), v.end());
  for (int32_t i = 0; i < n; ++i) {
    ids_out[i] = v[i].second;
    if (scores_out) scores_out[i] = v[i].first;
  }
  return FCG_OK;
}

}  // extern "C"
