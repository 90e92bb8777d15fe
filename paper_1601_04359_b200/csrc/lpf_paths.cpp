// lpf_paths.cpp -- host side of liblpf.so: paper "step 1".
//   * closed-form Bresenham rasteriser for the canonical half D (Eq. 13)
//   * prefix trie over all P_v, |dx|,|dy| <= m
//   * partition of the trie into work items and linearisation into the node program that
//     the eval kernel interprets
// No CUDA calls here.  Shares nothing with oracle/ (which rasterises incrementally).
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "lpf_internal.h"

namespace lpf {

// P_v for v in D, closed form (reading D2; "Bresenham [20]"):
// one pixel per major-axis step k = 0..n, n = max(|dx|,|dy|); the minor coordinate is
// round-half-up of k*|minor|/n, i.e. floor((2k|minor| + n) / (2n)); signs applied after.
int canonical_path(int dx, int dy, int16_t* xy) {
  const int ax = std::abs(dx), ay = std::abs(dy);
  const int sx = (dx > 0) - (dx < 0), sy = (dy > 0) - (dy < 0);
  const int n = std::max(ax, ay);
  xy[0] = 0;
  xy[1] = 0;
  for (int k = 1; k <= n; ++k) {
    int px, py;
    if (ax >= ay) {
      px = k;
      py = (2 * k * ay + ax) / (2 * ax);
    } else {
      py = k;
      px = (2 * k * ax + ay) / (2 * ay);
    }
    xy[2 * k] = (int16_t)(sx * px);
    xy[2 * k + 1] = (int16_t)(sy * py);
  }
  return n + 1;
}

static void build_trie(lpf_paths* p) {
  const int m = p->m;
  std::vector<Node>& nd = p->nodes;
  nd.clear();
  nd.push_back(Node{0, 0, -1, -1, -1, 1, 0, 0});
  std::vector<int16_t> xy(2 * (size_t)(m + 1));
  p->n_half = 0;
  p->sum_len = 0;
  for (int dy = 0; dy <= m; ++dy)
    for (int dx = -m; dx <= m; ++dx) {
      if (!in_half(dx, dy)) continue;
      const int len = canonical_path(dx, dy, xy.data());
      p->n_half += 1;
      p->sum_len += len;
      int cur = 0;
      for (int k = 1; k < len; ++k) {
        const int16_t a = xy[2 * k], b = xy[2 * k + 1];
        int c = nd[cur].first_child;
        while (c >= 0 && !(nd[c].a == a && nd[c].b == b)) c = nd[c].next_sibling;
        if (c < 0) {
          c = (int)nd.size();
          nd.push_back(Node{a, b, cur, -1, nd[cur].first_child, 1, nd[cur].depth + 1, 0});
          nd[cur].first_child = c;
        }
        cur = c;
      }
      nd[cur].terminal = 1;
    }
  // children are created after their parent, so a reverse sweep accumulates subtree sizes
  for (int i = (int)nd.size() - 1; i > 0; --i) nd[nd[i].parent].size += nd[i].size;
}

// ---- program emission ----------------------------------------------------------------------

static inline uint64_t make_entry(int m, int a, int b, uint32_t flags, int rslot, int sslot) {
  const uint32_t sh = (uint32_t)(a & 31);
  const uint32_t col = (uint32_t)((a >> 5) + E_COL_BIAS);   // arithmetic shift: floor(a / 32)
  const uint32_t x = sh | (col << E_COL_SHIFT) | ((uint32_t)b << E_B_SHIFT) | flags;
  const uint32_t cidx = (uint32_t)((b + m) * (2 * m + 1) + (a + m));
  const uint32_t y = cidx | ((uint32_t)rslot << E_RSLOT_SHIFT) | ((uint32_t)sslot << E_SSLOT_SHIFT);
  return (uint64_t)x | ((uint64_t)y << 32);
}

struct Emitter {
  const lpf_paths* p;
  const std::vector<Node>& nd;
  const std::vector<uint8_t>& cut;      // node is the root of a piece
  const std::vector<int32_t>& psize;    // nodes of the subtree that stay in the node's own piece
  Program& out;
  int max_slots = 0;

  uint32_t step_flags(int node, int prev) const {   // ADV / RELOAD of a direct descent prev -> node
    uint32_t f = 0;
    if (nd[node].b == nd[prev].b + 1) f |= E_ADV;
    if ((nd[node].a >> 5) != (nd[prev].a >> 5)) f |= E_RELOAD;
    return f;
  }

  // emits `node` and the part of its subtree inside the piece. src: 0 direct, 1 restore(rslot), 2 init.
  void emit(int node, int src, int rslot, int depth_slots) {
    std::vector<int> kids;
    for (int c = nd[node].first_child; c >= 0; c = nd[c].next_sibling)
      if (!cut[c]) kids.push_back(c);
    // heaviest child last: its descent frees the slot, so live slots <= log2(piece size) + 1
    std::stable_sort(kids.begin(), kids.end(), [&](int x, int y) { return psize[x] < psize[y]; });
    uint32_t flags = nd[node].terminal ? E_TERMINAL : 0u;
    if (src == 1) flags |= E_RESTORE;
    if (src == 2) flags |= E_INIT;
    if (src == 0) flags |= step_flags(node, nd[node].parent);
    int sslot = 0;
    if (kids.size() >= 2) {
      flags |= E_SAVE;
      sslot = depth_slots;
      max_slots = std::max(max_slots, depth_slots + 1);
    }
    const size_t at = out.entries.size();
    out.entries.push_back(make_entry(p->m, nd[node].a, nd[node].b, flags, rslot, sslot));
    out.skip.push_back(0);
    for (size_t i = 0; i < kids.size(); ++i) {
      if (kids.size() == 1) {
        emit(kids[i], 0, 0, depth_slots);
      } else if (i == 0) {
        emit(kids[i], 0, 0, depth_slots + 1);
      } else if (i + 1 < kids.size()) {
        emit(kids[i], 1, sslot, depth_slots + 1);
      } else {
        emit(kids[i], 1, sslot, depth_slots);      // last child: the slot is free again
      }
    }
    out.skip[at] = (uint32_t)(out.entries.size() - at - 1);
  }
};

static void sort_items(Program& pr) {
  const size_t n = pr.items.size() / 2;
  std::vector<std::pair<int64_t, int64_t>> v(n);
  for (size_t i = 0; i < n; ++i) v[i] = {pr.items[2 * i], pr.items[2 * i + 1]};
  std::stable_sort(v.begin(), v.end(), [](const std::pair<int64_t, int64_t>& a,
                                          const std::pair<int64_t, int64_t>& b) { return a.second > b.second; });
  for (size_t i = 0; i < n; ++i) {
    pr.items[2 * i] = v[i].first;
    pr.items[2 * i + 1] = v[i].second;
  }
}

static void build_trie_program(lpf_paths* p, int piece_nodes, Program& pr) {
  const std::vector<Node>& nd = p->nodes;
  const int N = (int)nd.size();
  std::vector<uint8_t> cut(N, 0);
  std::vector<int32_t> psize(N, 1);
  // greedy bottom-up partition: a node whose residual subtree reaches piece_nodes starts a piece
  for (int i = N - 1; i > 0; --i) {
    if (piece_nodes > 0 && psize[i] >= piece_nodes) cut[i] = 1;
    else psize[nd[i].parent] += psize[i];
  }
  cut[0] = 1;
  Emitter em{p, nd, cut, psize, pr};
  std::vector<int> chain;
  for (int r = 0; r < N; ++r) {
    if (!cut[r]) continue;
    const int64_t first = (int64_t)pr.entries.size();
    // chain root -> parent(r): recomputed per item, never counted, never saved
    chain.clear();
    for (int u = nd[r].parent; u >= 0; u = nd[u].parent) chain.push_back(u);
    std::reverse(chain.begin(), chain.end());
    for (size_t i = 0; i < chain.size(); ++i) {
      const int u = chain[i];
      const uint32_t f = (i == 0) ? E_INIT : em.step_flags(u, chain[i - 1]);
      pr.entries.push_back(make_entry(p->m, nd[u].a, nd[u].b, f, 0, 0));
      pr.skip.push_back(0);
    }
    em.emit(r, chain.empty() ? 2 : 0, 0, 0);
    pr.items.push_back(first);
    pr.items.push_back((int64_t)pr.entries.size() - first);
  }
  pr.n_slots = em.max_slots;
  sort_items(pr);
}

// LPF_NO_TRIE: one chain per path, no sharing ("one-path-per-warp" variant of the north star)
static void build_chain_program(lpf_paths* p, int piece_nodes, Program& pr) {
  const int m = p->m;
  std::vector<int16_t> xy(2 * (size_t)(m + 1));
  int64_t first = 0;
  for (int dy = 0; dy <= m; ++dy)
    for (int dx = -m; dx <= m; ++dx) {
      if (!in_half(dx, dy)) continue;
      const int len = canonical_path(dx, dy, xy.data());
      for (int k = 0; k < len; ++k) {
        uint32_t f = (k == 0) ? E_INIT : 0u;
        if (k > 0) {
          if (xy[2 * k + 1] == xy[2 * k - 1] + 1) f |= E_ADV;
          if ((xy[2 * k] >> 5) != (xy[2 * k - 2] >> 5)) f |= E_RELOAD;
        }
        if (k == len - 1) f |= E_TERMINAL;
        pr.entries.push_back(make_entry(m, xy[2 * k], xy[2 * k + 1], f, 0, 0));
        pr.skip.push_back(0);
      }
      const int64_t cur = (int64_t)pr.entries.size();
      if (piece_nodes > 0 && cur - first >= piece_nodes) {
        pr.items.push_back(first);
        pr.items.push_back(cur - first);
        first = cur;
      }
    }
  const int64_t cur = (int64_t)pr.entries.size();
  if (cur > first) {
    pr.items.push_back(first);
    pr.items.push_back(cur - first);
  }
  pr.n_slots = 0;
  sort_items(pr);
}

Program& get_program(lpf_paths* p, int piece_nodes, unsigned flags) {
  if (piece_nodes < 0) piece_nodes = 0;
  const std::pair<int, unsigned> key(piece_nodes, flags & LPF_NO_TRIE);
  auto it = p->programs.find(key);
  if (it != p->programs.end()) return it->second;
  Program& pr = p->programs[key];
  if (flags & LPF_NO_TRIE) build_chain_program(p, piece_nodes, pr);
  else build_trie_program(p, piece_nodes, pr);
  return pr;
}

int build_host_table(lpf_paths* p) {
  try {
    build_trie(p);
  } catch (const std::bad_alloc&) {
    return LPF_E_NOMEM;
  }
  return LPF_OK;
}

}  // namespace lpf

// ---- host-only C ABI entry points ------------------------------------------------------------

extern "C" const char* lpf_strerror(int code) {
  switch (code) {
    case LPF_OK: return "ok";
    case LPF_E_INVAL: return "invalid argument";
    case LPF_E_NOMEM: return "out of memory";
    case LPF_E_CUDA: return "CUDA runtime error";
    case LPF_E_UNSUPPORTED: return "unsupported shape";
    default: return "unknown error";
  }
}

extern "C" int lpf_paths_info(const lpf_paths* p, int64_t* n_half_vectors, int64_t* sum_path_len,
                              int64_t* n_trie_nodes, int* max_depth) {
  if (!p) return LPF_E_INVAL;
  if (n_half_vectors) *n_half_vectors = p->n_half;
  if (sum_path_len) *sum_path_len = p->sum_len;
  if (n_trie_nodes) *n_trie_nodes = (int64_t)p->nodes.size();
  if (max_depth) {
    int d = 0;
    for (const lpf::Node& n : p->nodes) d = std::max(d, (int)n.depth);
    *max_depth = d;
  }
  return LPF_OK;
}

extern "C" int lpf_paths_get(const lpf_paths* p, int dx, int dy, int16_t* xy, int cap, int* len) {
  if (!p || !xy || !len) return LPF_E_INVAL;
  const int m = p->m;
  if (dx < -m || dx > m || dy < -m || dy > m) return LPF_E_INVAL;
  const int n = std::max(std::abs(dx), std::abs(dy)) + 1;
  if (cap < n) return LPF_E_INVAL;
  if (lpf::in_half(dx, dy)) {
    lpf::canonical_path(dx, dy, xy);
  } else {
    // DESIGN.md reading D3: P_v = reverse(P_{-v}) + v
    std::vector<int16_t> t(2 * (size_t)n);
    lpf::canonical_path(-dx, -dy, t.data());
    for (int k = 0; k < n; ++k) {
      xy[2 * k] = (int16_t)(t[2 * (n - 1 - k)] + dx);
      xy[2 * k + 1] = (int16_t)(t[2 * (n - 1 - k) + 1] + dy);
    }
  }
  *len = n;
  return LPF_OK;
}

extern "C" int lpf_paths_program(lpf_paths* p, int piece_nodes, unsigned flags, uint64_t* entries,
                                 int64_t cap_entries, int64_t* n_entries, int64_t* items,
                                 int64_t cap_items, int64_t* n_items, int* n_slots) {
  if (!p || !n_entries || !n_items || !n_slots) return LPF_E_INVAL;
  try {
    lpf::Program& pr = lpf::get_program(p, piece_nodes, flags);
    *n_entries = (int64_t)pr.entries.size();
    *n_items = (int64_t)pr.items.size() / 2;
    *n_slots = pr.n_slots;
    if (entries) {
      if (cap_entries < *n_entries) return LPF_E_INVAL;
      std::memcpy(entries, pr.entries.data(), sizeof(uint64_t) * pr.entries.size());
    }
    if (items) {
      if (cap_items < *n_items) return LPF_E_INVAL;
      std::memcpy(items, pr.items.data(), sizeof(int64_t) * pr.items.size());
    }
  } catch (const std::bad_alloc&) {
    return LPF_E_NOMEM;
  }
  return LPF_OK;
}
