// Submatrix combination heuristic (section III-B3, Eq. 14): integer work on the
// HOST, upstream of a0 -- the paper runs it on one node's CPU cores, off the clock, and reuses the result for many
// MD steps.  Clusters of molecules are merged while Eq. 14 says the merged submatrix costs
// fewer cubic FLOPs than the two it replaces; candidates are found through the row entries of T_i itself and taken
// in sweeps over n_{j\i} = 0, 1, 2, ....  The serialisation of what the paper does "in parallel" is
// DESIGN.md reading 22: clusters ascending, candidates ascending, T_i updated at once, sweeps restarted until a
// whole round merges nothing.  The expensive part -- |R_i n R_j| -- is cached per pair and recomputed only when one
// of the two row sets changed, which does not alter the sequence of decisions.
#include <algorithm>
#include <unordered_map>
#include "common.cuh"

namespace {

struct PairInfo { int32_t ver_j, common; };

struct Cluster {
  std::vector<int32_t> rows, owners;     // sorted row set R_i (molecules); owners in merge order
  bool alive = true;
  int32_t ver = 0;                        // bumped whenever rows changes or the cluster dies
  int32_t cache_ver = 0;                  // version of rows the cache was filled for
  std::unordered_map<int32_t, PairInfo> cache;
};

int32_t count_common(const std::vector<int32_t> &a, const std::vector<int32_t> &b) {
  int32_t c = 0;
  size_t i = 0, j = 0;
  while (i < a.size() && j < b.size()) {
    if (a[i] < b[j]) ++i;
    else if (a[i] > b[j]) ++j;
    else { ++c; ++i; ++j; }
  }
  return c;
}

// Eq. 14 in exact integers (n <= 2^20 molecules -> cubes < 2^63)
bool merge_gain(int64_t ni, int64_t nj, int64_t common) {
  const int64_t m = ni + nj - common;
  return m * m * m < ni * ni * ni + nj * nj * nj;
}

}  // namespace

extern "C" nolsm_status nolsm_combine_submatrices(int32_t n_mol, const int32_t *row_ptr, const int32_t *col_idx,
                                                  int32_t *n_groups_out, int32_t *own_ptr, int32_t *own_idx,
                                                  int32_t *list_ptr, int32_t *list_idx, int64_t list_cap,
                                                  int64_t *list_len_out) {
  if (n_mol < 0 || !row_ptr || (n_mol > 0 && !col_idx) || !n_groups_out || !own_ptr || !own_idx || !list_ptr ||
      list_cap < 0 || (list_cap > 0 && !list_idx))
    return NOLSM_EINVAL;
  if (n_mol >= (1 << 20)) return NOLSM_EINVAL;
  std::vector<Cluster> cl((size_t)n_mol);
  std::vector<int32_t> owner_of((size_t)n_mol);
  for (int32_t i = 0; i < n_mol; ++i) {
    if (row_ptr[i + 1] < row_ptr[i]) return NOLSM_EINVAL;
    cl[i].rows.assign(col_idx + row_ptr[i], col_idx + row_ptr[i + 1]);
    for (size_t k = 0; k < cl[i].rows.size(); ++k) {
      const int32_t r = cl[i].rows[k];
      if (r < 0 || r >= n_mol || (k > 0 && r <= cl[i].rows[k - 1])) return NOLSM_EINVAL;   // ascending, in range
    }
    cl[i].owners.assign(1, i);
    owner_of[i] = i;
  }
  std::vector<int32_t> cand, merged;
  for (;;) {
    bool merged_any = false;
    size_t d_max = 0;
    for (const Cluster &c : cl)
      if (c.alive) d_max = std::max(d_max, c.rows.size());
    for (int32_t d = 0; d <= (int32_t)d_max; ++d) {
      for (int32_t i = 0; i < n_mol; ++i) {
        Cluster &ci = cl[i];
        if (!ci.alive) continue;
        // first filter: the clusters that own a row entry of T_i (snapshot at the start of the scan)
        cand.clear();
        for (int32_t m : ci.rows)
          if (owner_of[m] != i) cand.push_back(owner_of[m]);
        std::sort(cand.begin(), cand.end());
        cand.erase(std::unique(cand.begin(), cand.end()), cand.end());
        for (int32_t j : cand) {
          Cluster &cj = cl[j];
          if (!cj.alive || j == i) continue;
          if (ci.cache_ver != ci.ver) { ci.cache.clear(); ci.cache_ver = ci.ver; }
          auto it = ci.cache.find(j);
          if (it == ci.cache.end() || it->second.ver_j != cj.ver) {
            const PairInfo pi{cj.ver, count_common(ci.rows, cj.rows)};
            if (it == ci.cache.end()) it = ci.cache.emplace(j, pi).first; else it->second = pi;
          }
          const int32_t common = it->second.common;
          if ((int32_t)cj.rows.size() - common != d) continue;
          if (!merge_gain((int64_t)ci.rows.size(), (int64_t)cj.rows.size(), common)) continue;
          merged.resize(ci.rows.size() + cj.rows.size());
          merged.resize((size_t)(std::set_union(ci.rows.begin(), ci.rows.end(), cj.rows.begin(), cj.rows.end(),
                                                merged.begin()) - merged.begin()));
          ci.rows.swap(merged);
          ++ci.ver;
          for (int32_t m : cj.owners) owner_of[m] = i;
          ci.owners.insert(ci.owners.end(), cj.owners.begin(), cj.owners.end());
          cj.alive = false;
          ++cj.ver;
          std::vector<int32_t>().swap(cj.rows);
          std::vector<int32_t>().swap(cj.owners);
          cj.cache.clear();
          merged_any = true;
        }
      }
    }
    if (!merged_any) break;
  }
  // output: clusters ordered by their smallest owner, owners and rows ascending
  std::vector<std::pair<int32_t, int32_t>> order;
  for (int32_t i = 0; i < n_mol; ++i)
    if (cl[i].alive) {
      std::sort(cl[i].owners.begin(), cl[i].owners.end());
      order.emplace_back(cl[i].owners[0], i);
    }
  std::sort(order.begin(), order.end());
  int64_t list_len = 0;
  for (const auto &o : order) list_len += (int64_t)cl[o.second].rows.size();
  *n_groups_out = (int32_t)order.size();
  if (list_len_out) *list_len_out = list_len;
  if (list_len > list_cap) return NOLSM_ENOMEM;
  int32_t g = 0, op = 0;
  int64_t lp = 0;
  own_ptr[0] = 0;
  list_ptr[0] = 0;
  for (const auto &o : order) {
    const Cluster &c = cl[o.second];
    for (int32_t m : c.owners) own_idx[op++] = m;
    for (int32_t r : c.rows) list_idx[lp++] = r;
    ++g;
    own_ptr[g] = op;
    list_ptr[g] = (int32_t)lp;
  }
  return NOLSM_OK;
}

// Merged sparsity pattern of H0 and S ("row i is kept if H_ij != 0 or S_ij != 0"): the union of two
// block patterns given as host CSR arrays with ascending rows.  Host integer work, done once per pattern change.
extern "C" nolsm_status nolsm_union_pattern(int32_t n_mol, const int32_t *row_ptr_a, const int32_t *col_idx_a,
                                            const int32_t *row_ptr_b, const int32_t *col_idx_b, int32_t *row_ptr_u,
                                            int32_t *col_idx_u, int64_t cap, int64_t *nnzb_out) {
  if (n_mol < 0 || !row_ptr_a || !row_ptr_b || !row_ptr_u || cap < 0 || (cap > 0 && !col_idx_u)) return NOLSM_EINVAL;
  int64_t total = 0;
  for (int pass = 0; pass < 2; ++pass) {
    int64_t w = 0;
    for (int32_t i = 0; i < n_mol; ++i) {
      int32_t a = row_ptr_a[i], ae = row_ptr_a[i + 1], b = row_ptr_b[i], be = row_ptr_b[i + 1];
      if (ae < a || be < b) return NOLSM_EINVAL;
      if (pass == 1) row_ptr_u[i] = (int32_t)w;
      while (a < ae || b < be) {
        int32_t c;
        if (b >= be || (a < ae && col_idx_a[a] < col_idx_b[b])) c = col_idx_a[a++];
        else if (a >= ae || col_idx_b[b] < col_idx_a[a]) c = col_idx_b[b++];
        else { c = col_idx_a[a]; ++a; ++b; }
        if (pass == 1) col_idx_u[w] = c;
        ++w;
      }
    }
    if (pass == 0) {
      total = w;
      if (nnzb_out) *nnzb_out = total;
      if (total > cap || total > 0x7fffffff) return NOLSM_ENOMEM;
    } else {
      row_ptr_u[n_mol] = (int32_t)w;
    }
  }
  return NOLSM_OK;
}
