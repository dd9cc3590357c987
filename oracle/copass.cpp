// copass.cpp -- CPU oracle of the COPASS block-sort (Appendix A).  TEST INFRASTRUCTURE: see
// copass.h for who may use it, for the readings C1-C6 and for what pins it.  Plain single-threaded C++; every
// step below names the equation it restates.  Notation: m_lo = m-underbar, m_hi = m-bar, t_lo / t_hi the
// thresholds they belong to, mu_lo = mu, mu_hi = mu-bar, t_tilde, m_tilde, l as in the appendix.
#include "copass.h"

#include <algorithm>
#include <numeric>
#include <utility>
#include <vector>

namespace {

// card{j : S_j <= t} and card{j : S_j < t} of an ascending subarray (Eqs. A12, A13, A25, A26): binary searches
// ("can be computed through a binary search algorithm").
uint64_t card_le(const int64_t* S, uint64_t N, int64_t t) { return (uint64_t)(std::upper_bound(S, S + N, t) - S); }
uint64_t card_lt(const int64_t* S, uint64_t N, int64_t t) { return (uint64_t)(std::lower_bound(S, S + N, t) - S); }

uint64_t sum(const std::vector<uint64_t>& v) { return std::accumulate(v.begin(), v.end(), (uint64_t)0); }

}  // namespace

extern "C" int oc_copass_partition(const int64_t* keys, const uint64_t* start, const uint64_t* len, uint32_t k,
                                   uint64_t m, uint64_t* m_out, oc_copass_info* info) {
  if (!keys || !start || !len || !m_out || k == 0) return -1;
  uint64_t total = 0;
  for (uint32_t i = 0; i < k; ++i) total += len[i];
  if (m == 0 || m >= total) return -1;  // Eq. A4 / PAPER.md:464 (reading C1)
  auto S = [&](uint32_t i) { return keys + start[i]; };
  for (uint32_t i = 0; i < k; ++i)      // Eq. A5: each subarray ascending
    for (uint64_t j = 1; j < len[i]; ++j)
      if (S(i)[j - 1] > S(i)[j]) return -1;

  // Eqs. A14-A17: t_lo = min - 1, t_hi = max + 1, m_lo = 0, m_hi = N_i
  int64_t lo = INT64_MAX, hi = INT64_MIN;
  for (uint32_t i = 0; i < k; ++i)
    if (len[i]) {
      lo = std::min(lo, S(i)[0]);
      hi = std::max(hi, S(i)[len[i] - 1]);
    }
  int64_t t_lo = lo - 1, t_hi = hi + 1;
  std::vector<uint64_t> m_lo(k, 0), m_hi(len, len + k), mu_lo(k), mu_hi(k);
  uint32_t iterations = 0;

  for (;;) {
    // Eq. A19 holds here: sum m_lo < m < sum m_hi.
    // Eqs. A20-A21: the subarray with the widest open interval (lowest i among equals, reading C2)
    uint32_t l = 0;
    uint64_t widest = 0;
    for (uint32_t i = 0; i < k; ++i)
      if (m_hi[i] - m_lo[i] > widest) {
        widest = m_hi[i] - m_lo[i];
        l = i;
      }
    if (widest <= 1) {
      // ---- Sec. A3, condition A36: last step, case 1 ----
      std::vector<std::pair<int64_t, uint32_t>> C;  // Eq. A37 (reading C3): (S_{i, m_lo_i}, i) where m_hi = m_lo + 1
      for (uint32_t i = 0; i < k; ++i)
        if (m_hi[i] == m_lo[i] + 1) C.emplace_back(S(i)[m_lo[i]], i);
      std::sort(C.begin(), C.end());                 // Eq. A38
      const uint64_t d = m - sum(m_lo);              // Eq. A39
      for (uint32_t i = 0; i < k; ++i) m_out[i] = m_lo[i];           // Eq. A41
      for (uint64_t q = 0; q < d; ++q) m_out[C[q].second] += 1;      // Eqs. A40, A42
      if (info) *info = oc_copass_info{C[d - 1].first, iterations, 1};
      (void)t_lo;
      (void)t_hi;
      return 0;
    }
    ++iterations;
    const uint64_t m_tilde = (m_lo[l] + m_hi[l]) / 2;  // Eq. A22
    const int64_t t_tilde = S(l)[m_tilde];            // Eq. A23
    for (uint32_t i = 0; i < k; ++i) {
      mu_hi[i] = card_le(S(i), len[i], t_tilde);      // Eq. A25
      mu_lo[i] = card_lt(S(i), len[i], t_tilde);      // Eq. A26
    }
    const uint64_t sum_mu_lo = sum(mu_lo), sum_mu_hi = sum(mu_hi);
    if (sum_mu_lo <= m && m <= sum_mu_hi) {
      // ---- case 1 of the iteration, Eq. A29 -> Sec. A4: last step, case 2; t = t_tilde ----
      uint64_t d = m - sum_mu_lo;                     // Eq. A45
      for (uint32_t i = 0; i < k; ++i) {
        const uint64_t d_i = std::min(mu_hi[i] - mu_lo[i], d);  // Eqs. A46-A47 (reading C4)
        m_out[i] = mu_lo[i] + d_i;                    // Eq. A48
        d -= d_i;
      }
      if (info) *info = oc_copass_info{t_tilde, iterations, 2};
      return 0;
    }
    if (m < sum_mu_lo) {  // case 2, Eqs. A30-A32
      m_hi = mu_lo;
      t_hi = t_tilde;
    } else {              // case 3, Eqs. A33-A35
      m_lo = mu_hi;
      t_lo = t_tilde;
    }
  }
}

extern "C" int oc_copass_block_sort(int64_t* keys, uint32_t* vals, const uint64_t* N, uint32_t k,
                                    uint32_t max_extract, uint64_t* sub_start_out, uint64_t* sub_len_out,
                                    oc_copass_stats* stats) {
  if (!keys || !vals || !N || k == 0) return -1;
  oc_copass_stats st{};
  std::vector<uint64_t> block_off(k + 1, 0);
  for (uint32_t i = 0; i < k; ++i) block_off[i + 1] = block_off[i] + N[i];

  // the underlying sort, stable (reading C6), on keys[a .. a+n) with vals carried along
  auto sort_range = [&](int64_t* kk, uint32_t* vv, uint64_t n) {
    std::vector<uint64_t> order(n);
    std::iota(order.begin(), order.end(), (uint64_t)0);
    std::stable_sort(order.begin(), order.end(), [&](uint64_t a, uint64_t b) { return kk[a] < kk[b]; });
    std::vector<int64_t> ks(n);
    std::vector<uint32_t> vs(n);
    for (uint64_t j = 0; j < n; ++j) {
      ks[j] = kk[order[j]];
      vs[j] = vv[order[j]];
    }
    std::copy(ks.begin(), ks.end(), kk);
    std::copy(vs.begin(), vs.end(), vv);
  };

  // Fig. 6B: every block sorted by the underlying sort; the logical subarrays start out as the blocks
  std::vector<uint64_t> sub_start(block_off.begin(), block_off.begin() + k), sub_len(N, N + k), m_i(k);
  for (uint32_t i = 0; i < k; ++i) sort_range(keys + sub_start[i], vals + sub_start[i], sub_len[i]);

  std::vector<int64_t> aux_k;
  std::vector<uint32_t> aux_v;
  for (uint32_t b = 0; b < k && b < max_extract; ++b) {
    const uint64_t left_total = N[b];
    const uint64_t remaining = sum(sub_len);
    if (left_total == 0) continue;
    // Fig. 6C: left partitions of total size N_b under a common threshold
    if (left_total < remaining) {
      oc_copass_info info{};
      const int rc = oc_copass_partition(keys, sub_start.data(), sub_len.data(), k, left_total, m_i.data(), &info);
      if (rc != 0) return rc;
      ++st.partitions;
      st.iterations += info.iterations;
      (info.last_step == 1 ? st.last_step_1 : st.last_step_2) += 1;
    } else {
      m_i = sub_len;  // the last block: everything that is left (reading C5)
    }
    // Fig. 6D: left partitions -> auxiliary array, in subarray order
    aux_k.clear();
    aux_v.clear();
    for (uint32_t i = 0; i < k; ++i) {
      aux_k.insert(aux_k.end(), keys + sub_start[i], keys + sub_start[i] + m_i[i]);
      aux_v.insert(aux_v.end(), vals + sub_start[i], vals + sub_start[i] + m_i[i]);
    }
    st.aux_peak = std::max<uint64_t>(st.aux_peak, aux_k.size());
    // Fig. 6E: right partitions shifted to the right so that block b becomes free: packed from the end of
    // block b in subarray order; the last subarray first, so nothing is overwritten before it has moved
    std::vector<uint64_t> new_start(k);
    {
      uint64_t at = block_off[b + 1];
      for (uint32_t i = 0; i < k; ++i) {
        new_start[i] = at;
        at += sub_len[i] - m_i[i];
      }
    }
    for (uint32_t i = k; i-- > 0;) {
      const uint64_t from = sub_start[i] + m_i[i], cnt = sub_len[i] - m_i[i];
      if (cnt && new_start[i] != from) {
        std::copy_backward(keys + from, keys + from + cnt, keys + new_start[i] + cnt);
        std::copy_backward(vals + from, vals + from + cnt, vals + new_start[i] + cnt);
        st.moved += cnt;
      }
      sub_start[i] = new_start[i];
      sub_len[i] = cnt;
    }
    // Fig. 6E-F (reading C5): the auxiliary array, sorted, is what block b holds from now on
    sort_range(aux_k.data(), aux_v.data(), aux_k.size());
    std::copy(aux_k.begin(), aux_k.end(), keys + block_off[b]);
    std::copy(aux_v.begin(), aux_v.end(), vals + block_off[b]);
  }
  if (sub_start_out) std::copy(sub_start.begin(), sub_start.end(), sub_start_out);
  if (sub_len_out) std::copy(sub_len.begin(), sub_len.end(), sub_len_out);
  if (stats) *stats = st;
  return 0;
}
