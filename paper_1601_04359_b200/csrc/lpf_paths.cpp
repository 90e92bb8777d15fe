// lpf_paths.cpp -- host side of liblpf.so: paper "step 1".
//   * closed-form Bresenham rasteriser for the canonical half D (Eq. 13)
//   * prefix tries over all P_v, |dx|,|dy| <= m, one per octant in that octant's view coordinates
//   * partition of the tries into work items and linearisation into the node program that
//     the eval kernel interprets
// No CUDA calls here.  Shares nothing with oracle/ (which rasterises incrementally).
#include <algorithm>
#include <array>
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

// inserts the pixel list xy[1..len-1] (already in the trie's coordinates) below the root
static void trie_insert(std::vector<Node>& nd, const int16_t* xy, int len) {
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

static void build_trie(lpf_paths* p) {
  const int m = p->m;
  std::vector<Node> all;   // one trie over D in image coordinates: only its size is kept (lpf_paths_info)
  all.push_back(Node{0, 0, -1, -1, -1, 1, 0, 0});
  for (int o = 0; o < 4; ++o) {
    p->oct[o].clear();
    p->oct[o].push_back(Node{0, 0, -1, -1, -1, 1, 0, 0});
  }
  std::vector<int16_t> xy(2 * (size_t)(m + 1)), vxy(2 * (size_t)(m + 1));
  p->n_half = 0;
  p->sum_len = 0;
  for (int dy = 0; dy <= m; ++dy)
    for (int dx = -m; dx <= m; ++dx) {
      if (!in_half(dx, dy)) continue;
      const int len = canonical_path(dx, dy, xy.data());
      p->n_half += 1;
      p->sum_len += len;
      trie_insert(all, xy.data(), len);
      const int o = octant_of(dx, dy);
      for (int k = 0; k < len; ++k) {
        int av, bv;
        to_view(o, xy[2 * k], xy[2 * k + 1], &av, &bv);
        vxy[2 * k] = (int16_t)av;
        vxy[2 * k + 1] = (int16_t)bv;
      }
      trie_insert(p->oct[o], vxy.data(), len);
    }
  p->n_trie_nodes = (int64_t)all.size();
  // children are created after their parent, so a reverse sweep accumulates subtree sizes
  for (int o = 0; o < 4; ++o) {
    std::vector<Node>& nd = p->oct[o];
    for (int i = (int)nd.size() - 1; i > 0; --i) nd[nd[i].parent].size += nd[i].size;
  }
}

// ---- swap-delta node records ----------------------------------------
// The single prefix trie over D in IMAGE coordinates, in depth-first preorder; one 16-byte record per node:
//   [0] (a & 0xffff) | (b << 16)    pixel offset of the node
//   [1] (dx & 0xffff) | (dy << 16)  a canonical vector whose path runs through the node (its prefix IS the chain
//                                   root -> node, so the ancestors' pixels follow from Bresenham arithmetic)
//   [2] nodes in the subtree, self included (first child = index + 1, next sibling = index + [2])
//   [3] bits 0-19: (b+m)(2m+1)+(a+m) if the prefix is a whole path P_v, else 0xFFFFF; bits 20-23: 3 (sa+1) + (sb+1)
//       for the step (sa, sb) from the parent; bit 24: the node has a next sibling
void build_swap_records(const lpf_paths* p, std::vector<int32_t>& rec, std::vector<int32_t>& rrec, int64_t max_rev) {
  const int m = p->m;
  std::vector<Node> nd;
  nd.push_back(Node{0, 0, -1, -1, -1, 1, 0, 0});
  std::vector<int16_t> xy(2 * (size_t)(m + 1));
  for (int dy = 0; dy <= m; ++dy)
    for (int dx = -m; dx <= m; ++dx) {
      if (!in_half(dx, dy)) continue;
      trie_insert(nd, xy.data(), canonical_path(dx, dy, xy.data()));
    }
  const size_t N = nd.size();
  std::vector<int32_t> rep(N, 0);           // representative vector, packed; children are created after parents
  for (int i = (int)N - 1; i >= 0; --i) {
    if (nd[i].terminal) rep[i] = (int32_t)(((uint32_t)(uint16_t)nd[i].a) | ((uint32_t)(uint16_t)nd[i].b << 16));
    if (i > 0) {
      nd[nd[i].parent].size += nd[i].size;
      if (!nd[nd[i].parent].terminal) rep[nd[i].parent] = rep[i];
    }
  }
  rec.assign(4 * N, 0);
  std::vector<int32_t> pre(N, 0);                   // trie index -> preorder position
  std::vector<std::pair<int, int>> stack{{0, 0}};   // (trie index, has next sibling)
  int32_t at = 0;
  std::vector<int> kids;
  while (!stack.empty()) {
    const int u = stack.back().first, sib = stack.back().second;
    stack.pop_back();
    const int par = nd[u].parent;
    int step = 4;
    if (par >= 0) step = 3 * (nd[u].a - nd[par].a + 1) + (nd[u].b - nd[par].b + 1);
    const uint32_t cidx = nd[u].terminal ? (uint32_t)((nd[u].b + m) * (2 * m + 1) + (nd[u].a + m)) : 0xFFFFFu;
    rec[4 * (size_t)at + 0] = (int32_t)(((uint32_t)(uint16_t)nd[u].a) | ((uint32_t)(uint16_t)nd[u].b << 16));
    rec[4 * (size_t)at + 1] = rep[u];
    rec[4 * (size_t)at + 2] = nd[u].size;
    rec[4 * (size_t)at + 3] = (int32_t)(cidx | ((uint32_t)step << 20) | ((uint32_t)sib << 24));
    pre[u] = at;
    ++at;
    kids.clear();
    for (int c = nd[u].first_child; c >= 0; c = nd[c].next_sibling) kids.push_back(c);
    // popped in reverse push order: the first pushed child is emitted last and has no next sibling
    for (size_t k = 0; k < kids.size(); ++k) stack.push_back({kids[k], k == 0 ? 0 : 1});
  }

  // The REVERSED trie: for every node u its steps read backwards, u -> root, inserted as a
  // word over the 9 step codes.  A node of this trie at depth j is a walk of j steps back from the pixel that a segment
  // must contain; it is COMPLETE for the trie node u of depth j whose whole backward walk it is.  Walks of different
  // nodes share their beginnings, so testing the prefix root -> u of every u costs one pixel test per distinct backward
  // walk that is still in phase, not one walk per u.  One record per node in preorder:
  //   [0] (ra & 0xffff) | (rb << 16)  offset of the walk's end from the pixel (minus the sum of its steps)
  //   [1] preorder index of the trie node it is complete for, or -1
  //   [2] nodes in the subtree, self included   [3] bit 0: the node has a next sibling
  rrec.clear();
  struct RNode { int32_t child[9]; int32_t fwd; int16_t a, b; };
  std::vector<RNode> rn;
  RNode root;
  for (int k = 0; k < 9; ++k) root.child[k] = -1;
  root.fwd = 0; root.a = 0; root.b = 0;
  rn.push_back(root);
  bool too_big = false;
  for (size_t u = 1; u < N && !too_big; ++u) {
    int cur = 0;
    for (int w = (int)u; nd[w].parent >= 0; w = nd[w].parent) {
      const int par = nd[w].parent;
      const int sa = nd[w].a - nd[par].a, sb = nd[w].b - nd[par].b;
      const int code = 3 * (sa + 1) + (sb + 1);
      int c = rn[cur].child[code];
      if (c < 0) {
        if ((int64_t)rn.size() >= max_rev) { too_big = true; break; }
        RNode x;
        for (int k = 0; k < 9; ++k) x.child[k] = -1;
        x.fwd = -1;
        x.a = (int16_t)(rn[cur].a - sa);
        x.b = (int16_t)(rn[cur].b - sb);
        c = (int)rn.size();
        rn.push_back(x);
        rn[cur].child[code] = c;
      }
      cur = c;
    }
    if (!too_big) rn[cur].fwd = pre[u];
  }
  if (too_big) return;                               // the caller keeps the per-node walks for this table
  const size_t R = rn.size();
  std::vector<int32_t> rsize(R, 1);
  // subtree sizes by an explicit post-order
  std::vector<std::pair<int, int>> st2{{0, 0}};      // (node, next child code to look at)
  while (!st2.empty()) {
    auto& top = st2.back();
    int k = top.second;
    while (k < 9 && rn[top.first].child[k] < 0) ++k;
    if (k < 9) {
      top.second = k + 1;
      st2.push_back({rn[top.first].child[k], 0});
    } else {
      const int done = top.first;
      st2.pop_back();
      if (!st2.empty()) rsize[st2.back().first] += rsize[done];
    }
  }
  rrec.assign(4 * R, 0);
  std::vector<std::pair<int, int>> st3{{0, 0}};
  int32_t rat = 0;
  while (!st3.empty()) {
    const int u = st3.back().first, sib = st3.back().second;
    st3.pop_back();
    rrec[4 * (size_t)rat + 0] = (int32_t)(((uint32_t)(uint16_t)rn[u].a) | ((uint32_t)(uint16_t)rn[u].b << 16));
    rrec[4 * (size_t)rat + 1] = rn[u].fwd;
    rrec[4 * (size_t)rat + 2] = rsize[u];
    rrec[4 * (size_t)rat + 3] = sib;
    ++rat;
    kids.clear();
    for (int k = 0; k < 9; ++k)
      if (rn[u].child[k] >= 0) kids.push_back(rn[u].child[k]);
    for (size_t k = 0; k < kids.size(); ++k) st3.push_back({kids[k], k == 0 ? 0 : 1});
  }
}

// ---- program emission ----------------------------------------------------------------------

// balanced_word / balanced_rank (lpf_kernels.cuh) as tables: the host asks for them once per trie node
struct PatternTables {
  uint8_t ok[MAX_LEVEL + 1][1 << MAX_LEVEL];
  int8_t rank[MAX_LEVEL + 1][1 << MAX_LEVEL];
  PatternTables() {
    for (int K = 0; K <= MAX_LEVEL; ++K) {
      int r = 0;
      for (unsigned q = 0; q < (1u << MAX_LEVEL); ++q) {
        ok[K][q] = (q < (1u << K)) && balanced_word(q, K);
        rank[K][q] = (int8_t)(ok[K][q] ? r++ : -1);
      }
    }
  }
};
static const PatternTables& pattern_tables() {
  static const PatternTables t;
  return t;
}

struct Held {            // the row strip that is in the registers when an entry runs
  int b = -1, col = -1, plane = -1;
};

// Emits the entries of one octant.  Program styles:
//   level 0: one entry per node, window read from the plain bit plane
//   level K >= 1: shared memory holds one eroded plane per K-step pattern q instead of the plain plane: plane q at
//     (a, b) is the AND of the K + 1 pixels (a + j, b + s_1 + .. + s_j), s_j = bit j-1 of q.  Every path step is
//     (+1, 0) or (+1, +1), so any K + 1 consecutive nodes of a path are ONE window of one of the pattern planes:
//       - a run of nodes whose own masks are never needed (not terminal, one child in the piece) is cut into entries
//         of K + 1 nodes each,
//       - a run that ends early (at a terminal, a branching node or a leaf) is read "backwards": the window that ENDS
//         at its last node also covers some ancestors, which are already in the mask (AND is idempotent);
//     the nodes above depth K have no entry (no window ends there): every item starts with the window root .. depth K,
//     and the terminals above depth K are counted by shallow_kernel.
struct Emitter {
  int m, o, stride;
  int K, band_words;
  const signed char* slot_of;           // level K: rank of a balanced pattern -> plane slot of the item's class
  const std::vector<Node>& nd;
  const std::vector<uint8_t>& cut;      // node is the root of a piece
  const std::vector<int32_t>& psize;    // nodes of the subtree that stay in the node's own piece
  Program& out;
  int max_slots = 0;

  // the entry whose window ends at node `tail` and whose last `s` pixels are new nodes (1 <= s <= K + 1)
  uint64_t entry(int tail, int s, uint32_t flags, Held* held, int rslot, int sslot) const {
    int anchor = tail;
    uint32_t q = 0;
    for (int j = K; j >= 1; --j) {                   // step j of the window leads to its pixel j
      const int par = nd[anchor].parent;
      q |= (uint32_t)(nd[anchor].b - nd[par].b) << (j - 1);
      anchor = par;
    }
    const int a = nd[anchor].a, b = nd[anchor].b;
    const int plane = K > 0 ? (int)slot_of[pattern_tables().rank[K][q]] : -1;   // >= 0: the class holds every pattern of its paths
    const bool direct = !(flags & (E_RESTORE | E_INIT));
    if (!direct || held->b != b || held->col != (a >> 5) || held->plane != plane) flags |= E_RELOAD;
    held->b = b; held->col = a >> 5; held->plane = plane;
    const uint32_t off = (uint32_t)(b * stride + (a >> 5) + (K > 0 ? plane * band_words : 0));
    const uint32_t x = (uint32_t)(a & 31) | flags | (K > 0 ? E_ERODED : 0u) | (off << E_OFF_SHIFT);
    int ia, ib;
    from_view(o, nd[tail].a, nd[tail].b, &ia, &ib);
    const uint32_t cidx = (uint32_t)((ib + m) * (2 * m + 1) + (ia + m));
    (void)s;
    const uint32_t y = cidx | ((uint32_t)rslot << E_RSLOT_SHIFT) | ((uint32_t)sslot << E_SSLOT_SHIFT) | (q << E_Q_SHIFT);
    return (uint64_t)x | ((uint64_t)y << 32);
  }

  void kids_of(int node, std::vector<int>* kids) const {
    kids->clear();
    for (int c = nd[node].first_child; c >= 0; c = nd[c].next_sibling)
      if (!cut[c]) kids->push_back(c);
    // heaviest child last: its descent frees the slot, so live slots <= log2(piece size) + 1
    std::stable_sort(kids->begin(), kids->end(), [&](int x, int y) { return psize[x] < psize[y]; });
  }

  // emits `node` and the part of its subtree inside the piece. src: 0 direct, 1 restore(rslot), 2 init.
  // pend: ancestors of `node` (its chain from the root) that wait to be covered by the window of this entry.
  void emit(int node, int src, int rslot, int depth_slots, bool count_it, Held held, int pend) {
    std::vector<int> kids;
    kids_of(node, &kids);
    int tail = node, s = pend + 1;
    bool term = nd[node].terminal && count_it;
    while (s < K + 1 && !term && kids.size() == 1) { // the tail's own mask is never needed: take its only child in
      tail = kids[0];
      ++s;
      term = nd[tail].terminal;
      kids_of(tail, &kids);
    }
    uint32_t flags = term ? E_TERMINAL : 0u;
    if (src == 1) flags |= E_RESTORE;
    if (src == 2) flags |= E_INIT;
    int sslot = 0;
    if (kids.size() >= 2) {
      flags |= E_SAVE;
      sslot = depth_slots;
      max_slots = std::max(max_slots, depth_slots + 1);
    }
    const size_t at = out.entries.size();
    out.entries.push_back(entry(tail, s, flags, &held, rslot, sslot));
    out.skip.push_back(0);
    for (size_t i = 0; i < kids.size(); ++i) {
      if (kids.size() == 1) {
        emit(kids[i], 0, 0, depth_slots, true, held, 0);
      } else if (i == 0) {
        emit(kids[i], 0, 0, depth_slots + 1, true, held, 0);
      } else if (i + 1 < kids.size()) {
        emit(kids[i], 1, sslot, depth_slots + 1, true, held, 0);
      } else {
        emit(kids[i], 1, sslot, depth_slots, true, held, 0);   // last child: the slot is free again
      }
    }
    out.skip[at] = (uint32_t)(out.entries.size() - at - 1);
  }

  // one work item: the chain root -> parent(r), recomputed, never counted, never saved, then r and its piece
  void emit_item(int r, bool count_root) {
    std::vector<int> chain;
    for (int u = nd[r].parent; u >= 0; u = nd[u].parent) chain.push_back(u);
    std::reverse(chain.begin(), chain.end());
    Held held;
    bool started = false;
    int pend = 0;
    for (size_t i = 0; i < chain.size(); ++i) {
      if (++pend < K + 1) continue;
      out.entries.push_back(entry(chain[i], K + 1, started ? 0u : E_INIT, &held, 0, 0));
      out.skip.push_back(0);
      started = true;
      pend = 0;
    }
    emit(r, started ? 0 : 2, 0, 0, count_root, held, pend);
  }

  // the nodes at depth exactly K below `u` that belong to u's piece (level K: the items of a piece rooted above depth K)
  void at_depth_K(int u, std::vector<int>* found) const {
    if (nd[u].depth == K) { found->push_back(u); return; }
    for (int c = nd[u].first_child; c >= 0; c = nd[c].next_sibling)
      if (!cut[c]) at_depth_K(c, found);
  }
};

static void sort_items(Program& pr) {
  const size_t n = pr.items.size() / 4;
  std::vector<std::array<int64_t, 4>> v(n);
  for (size_t i = 0; i < n; ++i)
    v[i] = {pr.items[4 * i], pr.items[4 * i + 1], pr.items[4 * i + 2], pr.items[4 * i + 3]};
  std::stable_sort(v.begin(), v.end(),
                   [](const std::array<int64_t, 4>& a, const std::array<int64_t, 4>& b) { return a[1] > b[1]; });
  for (size_t i = 0; i < n; ++i)
    for (int k = 0; k < 4; ++k) pr.items[4 * i + k] = v[i][k];
}

// marks the entries whose mask is never needed on its own and whose successor is a direct child (E_PAIR)
static void mark_pairs(Program& pr, int64_t first) {
  const int64_t end = (int64_t)pr.entries.size();
  for (int64_t k = first; k + 1 < end; ++k) {
    const uint32_t x = (uint32_t)pr.entries[k], xn = (uint32_t)pr.entries[k + 1];
    if (!(x & (E_TERMINAL | E_SAVE)) && !(xn & (E_INIT | E_RESTORE))) pr.entries[k] |= E_PAIR;
  }
}

static void push_item(Program& pr, int64_t first, int o) {
  mark_pairs(pr, first);
  pr.items.push_back(first);
  pr.items.push_back((int64_t)pr.entries.size() - first);
  pr.items.push_back(o);
  pr.items.push_back(0);
}

static void push_item_c(Program& pr, int64_t first, int o, int cls) {
  push_item(pr, first, o);
  pr.items.back() = cls;
}

// partitions one trie into pieces and emits its items
static void emit_trie(const lpf_paths* p, int o, const std::vector<Node>& nd, int piece_nodes, Program& pr,
                      const signed char* slot_of, int cls, int band_words, int K) {
  const int N = (int)nd.size();
  std::vector<uint8_t> cut(N, 0);
  std::vector<int32_t> psize(N, 1);
  // greedy bottom-up partition: a node whose residual subtree reaches piece_nodes starts a piece
  for (int i = N - 1; i > 0; --i) {
    if (piece_nodes > 0 && psize[i] >= piece_nodes) cut[i] = 1;
    else psize[nd[i].parent] += psize[i];
  }
  cut[0] = 1;
  Emitter em{p->m, o, pr.stride[o], K, band_words, slot_of, nd, cut, psize, pr};
  std::vector<int> starts;
  for (int r = 0; r < N; ++r) {
    if (!cut[r]) continue;
    if (nd[r].depth < K) {
      // a piece rooted above depth K: no window ends up there, so each of its nodes at depth K opens an item
      // (terminals above depth K are counted by shallow_kernel)
      starts.clear();
      em.at_depth_K(r, &starts);
      for (int d : starts) {
        const int64_t f = (int64_t)pr.entries.size();
        em.emit_item(d, true);
        push_item_c(pr, f, o, cls);
      }
      continue;
    }
    if (r == 0 && o != 0 && psize[0] == 1) continue;   // plain program: v = 0 is counted in octant 0 only
    const int64_t first = (int64_t)pr.entries.size();
    em.emit_item(r, !(r == 0 && o != 0));
    push_item_c(pr, first, o, cls);
  }
  pr.n_slots = std::max(pr.n_slots, em.max_slots);
}

// Level K >= 1: the vectors of an octant (those of at least K steps), sorted by slope, are cut into CLASSES whose paths
// use at most pr.n_planes step patterns between them (a digital straight segment has at most K + 1 patterns of length K,
// neighbouring slopes share most of them); every class gets its own prefix trie.  The short common trunk of the octant
// is walked once per class instead of once: a fraction of a percent of the entries.
static void build_class_tries(const lpf_paths* p, int o, int piece_nodes, Program& pr) {
  const int Kmax = pr.K;
  const std::vector<Node>& nd = p->oct[o];
  const int N = (int)nd.size();
  // patterns of the last K steps at every node, and the union over the path root -> node, for the level in use
  std::vector<uint8_t> pat(N, 0);
  std::vector<uint64_t> pathset(N, 0);
  int K = 0;
  auto patterns_of_level = [&](int level) {
    K = level;
    pat[0] = 0;
    pathset[0] = 0;
    for (int i = 1; i < N; ++i) {
      const int par = nd[i].parent;
      pat[i] = (uint8_t)((pat[par] >> 1) | ((nd[i].b - nd[par].b) << (K - 1)));
      pathset[i] = pathset[par];
      if (nd[i].depth >= K) pathset[i] |= 1ull << pattern_tables().rank[K][pat[i]];
    }
  };
  // the vectors of fewer than Kmax steps are counted by shallow_kernel, whatever the level of their class would be
  std::vector<int> terms;
  for (int i = 0; i < N; ++i)
    if (nd[i].terminal && nd[i].depth >= Kmax) terms.push_back(i);
  std::sort(terms.begin(), terms.end(), [&](int x, int y) {          // by slope b / a, then by length
    const long long l = (long long)nd[x].b * nd[y].a, r = (long long)nd[y].b * nd[x].a;
    if (l != r) return l < r;
    return nd[x].a < nd[y].a;
  });
  std::vector<int16_t> vxy(2 * (size_t)(p->m + 1));
  // shared memory of one image: the n_planes + 1 full-height bands the geometry reserved.  A class only needs the rows
  // its paths reach (band_rows + the largest b'), so a class of shallow slopes has room for more planes -- wider
  // classes, more units per key, fewer keys (pr.widen; not when the keys are few already: lpf_api.cu).  Where even
  // the patterns of ONE path do not fit at level Kmax (steep slopes of a template that is large against the image: a
  // plane is band_rows + m rows), the class takes the highest level that leaves room for them.
  const long long budget = (long long)(pr.n_planes + 1) * pr.band_words[o];
  auto room_at = [&](int bmax_c, int level, int* rows_out, int* bw_out) {
    const int rows = std::min(pr.band_rows + p->m, pr.band_rows + bmax_c + 1);
    const int bw = (rows * pr.stride[o] + 3) / 4 * 4;
    if (rows_out) *rows_out = rows;
    if (bw_out) *bw_out = bw;
    const int cap = pr.widen ? MAX_PATTERNS : std::max(pr.n_planes, 2);
    return (int)std::min<long long>({(long long)cap, (long long)balanced_count(level), budget / bw - 1});
  };
  size_t t0 = 0;
  while (t0 < terms.size()) {
    // the level of the class: the highest at which the patterns of one path fit (K + 1 of them)
    int level = Kmax;
    for (; level > 1; --level) {
      const int room = room_at(nd[terms[t0]].b, level, nullptr, nullptr);
      if (room >= std::min(balanced_count(level), p->path_patterns[level])) break;
    }
    if (level != K) patterns_of_level(level);
    uint64_t set = 0;
    size_t t1 = t0;
    int bmax = 0, rows_c = 0, bw_c = 0;
    while (t1 < terms.size()) {
      const uint64_t ns = set | pathset[terms[t1]];
      const int bm = std::max(bmax, (int)nd[terms[t1]].b);
      int rows = 0, bw = 0;
      const int room = room_at(bm, K, &rows, &bw);
      if (__builtin_popcountll(ns) > room) break;
      set = ns;
      bmax = bm;
      rows_c = rows;
      bw_c = bw;
      ++t1;
    }
    if (t1 == t0) return;                                  // cannot happen: level 1 has two patterns and two planes fit
    Program::Class c;
    c.octant = o;
    c.rows = rows_c;
    c.band_words = bw_c;
    c.level = K;
    std::memset(c.slot_of, -1, sizeof(c.slot_of));
    std::memset(c.pattern, 0, sizeof(c.pattern));
    for (unsigned q = 0; q < (1u << K); ++q) {
      if (!pattern_tables().ok[K][q]) continue;
      const int rank = pattern_tables().rank[K][q];
      if (!((set >> rank) & 1ull)) continue;
      c.slot_of[rank] = (signed char)c.n;
      c.pattern[c.n++] = (int)q;
    }
    std::vector<Node> cnd;
    cnd.push_back(Node{0, 0, -1, -1, -1, 1, 0, 0});
    for (size_t t = t0; t < t1; ++t) {
      int len = 0;
      for (int u = terms[t]; u >= 0; u = nd[u].parent) ++len;
      int k = len;
      for (int u = terms[t]; u >= 0; u = nd[u].parent) {
        --k;
        vxy[2 * k] = nd[u].a;
        vxy[2 * k + 1] = nd[u].b;
      }
      trie_insert(cnd, vxy.data(), len);
    }
    for (int i = (int)cnd.size() - 1; i > 0; --i) cnd[cnd[i].parent].size += cnd[i].size;
    const int cls = (int)pr.classes.size();
    pr.classes.push_back(c);
    emit_trie(p, o, cnd, piece_nodes, pr, pr.classes[cls].slot_of, cls, bw_c, K);
    t0 = t1;
  }
}

static void build_trie_program(lpf_paths* p, int piece_nodes, Program& pr) {
  for (int o = 0; o < 4; ++o) {
    if (pr.K == 0) emit_trie(p, o, p->oct[o], piece_nodes, pr, nullptr, 0, 0, 0);
    else build_class_tries(p, o, piece_nodes, pr);
  }
  sort_items(pr);
}

// The highest level (<= MAX_LEVEL) at which every window of every path is a balanced word, and for every level the
// largest number of different patterns on one path (a class needs that many planes at least; K + 1 for a digital
// straight segment).
static void analyse_levels(lpf_paths* p) {
  int ok = MAX_LEVEL;
  for (int o = 0; o < 4; ++o) {
    const std::vector<Node>& nd = p->oct[o];
    std::vector<uint8_t> pat(nd.size(), 0);                // last MAX_LEVEL steps, newest in the top bit
    for (size_t i = 1; i < nd.size(); ++i) {
      const int par = nd[i].parent;
      pat[i] = (uint8_t)((pat[par] >> 1) | ((nd[i].b - nd[par].b) << (MAX_LEVEL - 1)));
      for (int K = 2; K <= std::min<int>(ok, nd[i].depth); ++K)
        if (!pattern_tables().ok[K][(unsigned)pat[i] >> (MAX_LEVEL - K)]) ok = K - 1;
    }
  }
  p->level_ok = ok;
  for (int K = 0; K <= MAX_LEVEL; ++K) p->path_patterns[K] = 0;
  for (int K = 1; K <= ok; ++K)
    for (int o = 0; o < 4; ++o) {
      const std::vector<Node>& nd = p->oct[o];
      std::vector<uint8_t> pat(nd.size(), 0);
      std::vector<uint64_t> pathset(nd.size(), 0);
      for (size_t i = 1; i < nd.size(); ++i) {
        const int par = nd[i].parent;
        pat[i] = (uint8_t)((pat[par] >> 1) | ((nd[i].b - nd[par].b) << (K - 1)));
        pathset[i] = pathset[par];
        if (nd[i].depth >= K) pathset[i] |= 1ull << pattern_tables().rank[K][pat[i]];
        if (nd[i].terminal) p->path_patterns[K] = std::max(p->path_patterns[K], __builtin_popcountll(pathset[i]));
      }
    }
}

// the terminals above depth K of every octant trie, with their paths as step patterns (level K only)
void shallow_terminals(const lpf_paths* p, int K, ShallowList* out) {
  std::memset(out, 0, sizeof(*out));
  std::memset(out->node, -1, sizeof(out->node));
  const int m = p->m;
  for (int o = 0; o < 4; ++o) {
    const std::vector<Node>& nd = p->oct[o];
    for (int i = 0; i < (int)nd.size(); ++i) {
      if (nd[i].depth >= K || !nd[i].terminal) continue;
      unsigned steps = 0;
      for (int u = i; nd[u].parent >= 0; u = nd[u].parent)
        steps |= (unsigned)(nd[u].b - nd[nd[u].parent].b) << (nd[u].depth - 1);
      int ia, ib;
      from_view(o, nd[i].a, nd[i].b, &ia, &ib);
      if (out->n[o] >= MAX_SHALLOW) continue;            // cannot happen: K <= MAX_LEVEL
      const int k = out->n[o]++;
      out->cidx[o][k] = (ib + m) * (2 * m + 1) + (ia + m);
      out->node[o][shallow_base(nd[i].depth) + pattern_tables().rank[nd[i].depth][steps]] = (signed char)k;
    }
  }
}

// LPF_NO_TRIE: one chain per path, no sharing ("one-path-per-warp" variant of the north star).  An item opens with the
// root pixel (its only INIT entry, saved in slot 0); every path restores that mask and walks its pixels 1..n.
static void build_chain_program(lpf_paths* p, int piece_nodes, Program& pr) {
  const int m = p->m;
  std::vector<int16_t> xy(2 * (size_t)(m + 1));
  const uint32_t cidx0 = (uint32_t)(m * (2 * m + 1) + m);
  for (int o = 0; o < 4; ++o) {
    int64_t first = -1;
    bool zero_done = false;
    const int stride = pr.stride[o];
    for (int dy = 0; dy <= m; ++dy)
      for (int dx = -m; dx <= m; ++dx) {
        if (!in_half(dx, dy) || octant_of(dx, dy) != o) continue;
        if (first < 0) {                                   // open an item: the root pixel, saved in slot 0
          first = (int64_t)pr.entries.size();
          uint32_t x = E_INIT | E_RELOAD | E_SAVE;
          if (o == 0 && !zero_done) { x |= E_TERMINAL; zero_done = true; }   // v = 0 is counted once
          pr.entries.push_back((uint64_t)x | ((uint64_t)cidx0 << 32));
          pr.skip.push_back(0);
        }
        const int len = canonical_path(dx, dy, xy.data());
        int pa = 0, pb = 0;
        for (int k = 1; k < len; ++k) {
          int a, b;
          to_view(o, xy[2 * k], xy[2 * k + 1], &a, &b);
          uint32_t f = (k == 1) ? (E_RESTORE | E_RELOAD) : 0u;
          if (k > 1 && (b != pb || (a >> 5) != (pa >> 5))) f |= E_RELOAD;
          if (k == len - 1) f |= E_TERMINAL;
          const uint32_t off = (uint32_t)(b * stride + (a >> 5));
          const uint32_t x = (uint32_t)(a & 31) | f | (off << E_OFF_SHIFT);
          const uint32_t cidx = (uint32_t)((dy + m) * (2 * m + 1) + (dx + m));
          pr.entries.push_back((uint64_t)x | ((uint64_t)cidx << 32));   // restore slot 0
          pr.skip.push_back(0);
          pa = a;
          pb = b;
        }
        if (piece_nodes > 0 && (int64_t)pr.entries.size() - first >= piece_nodes) {
          push_item(pr, first, o);
          first = -1;
        }
      }
    if (first >= 0) push_item(pr, first, o);
  }
  pr.n_slots = 1;
  sort_items(pr);
}

// LPF_S2: two-point probability (Eq. 6).  Every vector is a 2-pixel "path" {0, v}: the root window is
// saved once per item and every vector restores it, ANDs the window at v and counts.  Items of about piece_nodes vectors.
static void build_s2_program(lpf_paths* p, int piece_nodes, Program& pr) {
  const int m = p->m;
  if (piece_nodes <= 0) piece_nodes = 1 << 30;
  for (int o = 0; o < 4; ++o) {
    const int stride = pr.stride[o];
    int64_t first = -1;
    int in_item = 0;
    bool zero_done = false;
    for (int dy = 0; dy <= m; ++dy)
      for (int dx = -m; dx <= m; ++dx) {
        if (!in_half(dx, dy) || octant_of(dx, dy) != o) continue;
        if (first < 0) {                                   // open an item: the root pixel, saved in slot 0
          first = (int64_t)pr.entries.size();
          uint32_t x = E_INIT | E_RELOAD | E_SAVE;
          const bool count_zero = (o == 0 && !zero_done);  // v = 0 is counted once, in octant 0
          if (count_zero) { x |= E_TERMINAL; zero_done = true; }
          const uint32_t cidx0 = (uint32_t)(m * (2 * m + 1) + m);
          pr.entries.push_back((uint64_t)x | ((uint64_t)cidx0 << 32));
          pr.skip.push_back(0);
          in_item = 0;
        }
        if (dx == 0 && dy == 0) continue;
        int a, b;
        to_view(o, dx, dy, &a, &b);
        const uint32_t off = (uint32_t)(b * stride + (a >> 5));
        const uint32_t x = (uint32_t)(a & 31) | E_RESTORE | E_RELOAD | E_TERMINAL | (off << E_OFF_SHIFT);
        const uint32_t cidx = (uint32_t)((dy + m) * (2 * m + 1) + (dx + m));
        pr.entries.push_back((uint64_t)x | ((uint64_t)cidx << 32));   // restore slot 0, save slot unused
        pr.skip.push_back(0);
        if (++in_item >= piece_nodes) {
          pr.items.push_back(first);
          pr.items.push_back((int64_t)pr.entries.size() - first);
          pr.items.push_back(o);
          pr.items.push_back(0);
          first = -1;
        }
      }
    if (first >= 0) {
      pr.items.push_back(first);
      pr.items.push_back((int64_t)pr.entries.size() - first);
      pr.items.push_back(o);
      pr.items.push_back(0);
    }
  }
  pr.n_slots = 1;
  sort_items(pr);
}

Program& get_program(lpf_paths* p, int piece_nodes, unsigned flags, int stride03, int stride12, int K, int n_planes,
                     int bw03, int bw12, int band_rows, bool widen) {
  if (piece_nodes < 0) piece_nodes = 0;
  const unsigned kind = (flags & LPF_S2) ? LPF_S2 : (flags & LPF_NO_TRIE);
  if (kind != 0) K = 0;                                    // the eroded planes serve the trie program only
  if (K == 0) bw03 = bw12 = n_planes = band_rows = 0;
  const std::tuple<int, unsigned, int, int, int, int, int> key(piece_nodes, kind, stride03, stride12,
                                                               1000000 * (widen ? 1 : 0) + 100000 * band_rows + 100 * K + n_planes, bw03, bw12);
  auto it = p->programs.find(key);
  if (it != p->programs.end()) return it->second;
  Program& pr = p->programs[key];
  pr.stride[0] = pr.stride[3] = stride03;
  pr.stride[1] = pr.stride[2] = stride12;
  pr.K = K;
  pr.n_planes = n_planes;
  pr.band_rows = band_rows;
  pr.widen = widen;
  pr.band_words[0] = pr.band_words[3] = bw03;
  pr.band_words[1] = pr.band_words[2] = bw12;
  if (flags & LPF_S2) build_s2_program(p, piece_nodes, pr);
  else if (flags & LPF_NO_TRIE) build_chain_program(p, piece_nodes, pr);
  else build_trie_program(p, piece_nodes, pr);
  return pr;
}

void drop_program(lpf_paths* p, const Program* pr) {
  for (auto it = p->programs.begin(); it != p->programs.end(); ++it)
    if (&it->second == pr) {
      if (!pr->d_entries) p->programs.erase(it);
      return;
    }
}

int build_host_table(lpf_paths* p) {
  try {
    build_trie(p);
    analyse_levels(p);
  } catch (const std::bad_alloc&) {
    return LPF_E_NOMEM;
  }
  return LPF_OK;
}

}  // namespace lpf

// ---- geometry (host only) ---------------------------------------------

#include "lpf_kernels.cuh"

namespace lpf {

static bool choose_geom_fixed(int m, int H, int W, int B, int max_smem, int tx, int ty, int cta_warps, int K,
                              int min_planes, Geom* out);

// Resident warps per SM of a geometry once the CTA is made of teams (lpf_api.cu picks the team count with the
// occupancy API; this is the same search on a model: 64 registers per thread, i.e. at most 1024 threads per SM).
// max_teams: teams that can find work on one key (a small trie has few pieces).
static int resident_warps(const Geom& g, int max_smem, int max_teams, int* teams) {
  const int ctas_smem = std::min(32, (max_smem + 1024) / (g.smem_bytes + 1024));
  int best = 0;
  const int nt_max = std::max(1, std::min(g.threads > 32 ? 15 : 32, max_teams));   // named barriers 1 .. 15
  for (int nt = 1; nt * g.threads <= EVAL_CTA_MAX_THREADS && nt <= nt_max; ++nt) {
    const int ctas = std::min(ctas_smem, 1024 / (nt * g.threads));
    const int warps = ctas * nt * (g.threads / 32);
    if (warps > best) { best = warps; if (teams) *teams = nt; }
  }
  return best;
}

// Relative cost of a geometry: program entries at level K (counted on the tries of m = 64 .. 256: 1.9 : 1 : 0.70 :
// 0.57 : 0.47 : 0.40 : 0.35 for K = 0 .. 6; a little is added for the higher levels, whose entries reload their row
// strip more often, and for pattern classes, each of which walks the trunk of its octant again)
// over the throughput at the resident warps (measured on config 3: 8 warps 0.57, 16 warps 0.87, 24 warps 0.985 of
// the rate at 32).
static double geom_cost(const Geom& g, int max_smem, int max_teams) {
  static const double entries[MAX_LEVEL + 1] = {1.9, 1.0, 0.73, 0.61, 0.50, 0.44, 0.39};
  const int w = resident_warps(g, max_smem, max_teams, nullptr);
  double rate;
  if (w >= 32) rate = 1.0;
  else if (w >= 24) rate = 0.985 + 0.015 * (w - 24) / 8.0;
  else if (w >= 16) rate = 0.87 + 0.115 * (w - 16) / 8.0;
  else if (w >= 8) rate = 0.57 + 0.30 * (w - 8) / 8.0;
  else rate = 0.57 * w / 8.0;
  const double classes = (g.K > 0 && g.v[0].n_planes < balanced_count(g.K)) ? 1.03 : 1.0;
  // classes of mixed levels (fewer full-height planes than the K + 1 patterns of a path): the steepest class runs at
  // level n_planes - 1, the shallow ones at K
  const int k_steep = g.K > 0 ? std::max(1, std::min(g.K, g.v[0].n_planes - 1)) : 0;
  return 0.5 * (entries[g.K] + entries[k_steep]) * classes / std::max(rate, 1e-3);
}

// teams that find work on one key: two pieces of at least 256 trie nodes each per team and octant
int max_teams_of(const lpf_paths* p) {
  long long n_nodes = 0;
  for (int o = 0; o < 4; ++o) n_nodes += (long long)p->oct[o].size();
  return (int)std::max<long long>(1, std::min<long long>(32, n_nodes / 4 / 512));
}

// erosion level and team size: the cheapest by geom_cost.  Small teams come first -- two warps, then one, four, eight
// (measured: config 3 3.73 / 3.76 / 3.89 / 3.78 ms, config 4 2.66 / 2.65 / 2.73 / 2.86 ms, 300 x 300 with m = 299
// 4.10 / 5.42 / 4.57 / 4.57 ms: small keys balance better and leave room for a higher level); a later candidate or a
// lower level must win by more than 3 %.
bool choose_geom(int m, int H, int W, int B, int max_smem, int cta_smem, int tx, int ty, int cta_warps, int max_level,
                 int max_teams, const int* path_patterns, Geom* out) {
  cta_smem = cta_smem > 0 ? std::min(cta_smem, max_smem) : max_smem;   // lpf_set_shared_memory
  max_level = std::max(0, std::min({max_level, MAX_LEVEL, m}));   // the caller caps it at the table's level_ok
  double best = 0;
  bool found = false;
  static const int team_warps[4] = {2, 1, 4, 8};
  for (int K = max_level; K >= 0; --K)
    for (int ci = 0; ci < 4; ++ci) {
      const bool fixed = cta_warps >= 1 && cta_warps <= 8;   // lpf_set_tile: that team size only
      if (fixed && ci > 0) break;
      const int cw = fixed ? cta_warps : team_warps[ci];
      Geom g;
      if (!choose_geom_fixed(m, H, W, B, cta_smem, tx, ty, cw, K, path_patterns[K], &g)) continue;
      const double c = geom_cost(g, max_smem, max_teams);
      if (!found || c < best * 0.97) {
        best = c;
        *out = g;
        found = true;
      }
    }
  return found;
}

static bool choose_geom_fixed(int m, int H, int W, int B, int max_smem, int tx, int ty, int cta_warps, int K,
                              int min_planes, Geom* out) {
  Geom g;
  std::memset(&g, 0, sizeof(g));
  g.H = H; g.W = W; g.m = m; g.K = K;
  const int planes_all = K > 0 ? balanced_count(K) : 0;
  const int wc_max = (std::max(H, W) + 31) / 32;
  if (tx > 0 && ty > 0) {
    g.TX = tx; g.TY = ty;
  } else {                                       // thread tile of 16 words
    g.TX = wc_max >= 16 ? 16 : (wc_max >= 8 ? 8 : 4);
    g.TY = 16 / g.TX;
  }
  if (cta_warps < 1 || cta_warps > 8) cta_warps = 8;
  const int rows_per_warp = 32 * g.TY;
  int strips_max = 0, hv_max = 0;
  for (int o = 0; o < 4; ++o) {
    ViewGeom& v = g.v[o];
    const bool tr = (o == 1 || o == 2);
    v.Hv = tr ? W : H;
    v.Wv = tr ? H : W;
    v.Wc = (v.Wv + 31) / 32;
    v.n_strips = (v.Wc + g.TX - 1) / g.TX;
    v.stride = v.n_strips * g.TX + m / 32 + 1;
    if (!(v.stride & 1)) v.stride += 1;          // odd: 32 consecutive rows of one column hit 32 banks
    strips_max = std::max(strips_max, v.n_strips);
    hv_max = std::max(hv_max, v.Hv);
  }
  g.SB = std::min(strips_max, cta_warps);
  int row_blocks = std::max(1, cta_warps / g.SB);
  const int max_blocks = (hv_max + rows_per_warp - 1) / rows_per_warp;
  row_blocks = std::min(row_blocks, max_blocks);
  const int row_blocks0 = row_blocks;
  // first choice: bands low enough that every class has room for the patterns of one path at level K; where no band
  // is (a template that is large against the image), the steep classes run at lower levels (build_class_tries)
  bool mixed = false;
  for (;;) {
    g.band_rows = rows_per_warp * row_blocks;
    g.wpi = g.SB * row_blocks;
    int bw_max = 0;
    for (int o = 0; o < 4; ++o) {
      ViewGeom& v = g.v[o];
      v.n_bands = (v.Hv + g.band_rows - 1) / g.band_rows;
      v.band_words = ((g.band_rows + m) * v.stride + 3) / 4 * 4;
      v.plane_words = ((v.n_bands * g.band_rows + m) * v.stride + 3) / 4 * 4 + 4;
      v.view_words = v.plane_words;                         // only the plain view is kept in HBM
      bw_max = std::max(bw_max, v.band_words);
    }
    // level K: as many planes per pattern class as fit beside the plain band they are derived from (all balanced
    // patterns if possible); a class needs room for the patterns of one path (K + 1 for a digital straight segment)
    int n_planes = 0;
    if (K > 0) {
      n_planes = std::min(planes_all, (int)(((size_t)max_smem - 1024) / ((size_t)bw_max * 4)) - 1);
      const int need = mixed ? 2 : std::min(planes_all, std::max(min_planes, K + 1));   // level 1: two patterns
      if (n_planes < need) n_planes = -1;
    }
    if (n_planes >= 0) {
      for (int o = 0; o < 4; ++o) {
        g.v[o].n_planes = n_planes;
        g.v[o].band_pitch = (n_planes ? n_planes + 1 : 1) * g.v[o].band_words;
      }
      const size_t per_image = (size_t)(n_planes ? n_planes + 1 : 1) * bw_max * 4;   // shared memory holds the G bands
      int G = std::max(1, cta_warps / g.wpi);
      G = std::min(G, std::max(B, 1));
      G = (int)std::min<size_t>((size_t)G, ((size_t)max_smem - 1024) / per_image);
      g.G = std::max(G, 1);
      g.NT = 1;
      g.threads = g.G * g.wpi * 32;
      g.smem_bytes = (int)(g.G * per_image);
      break;
    }
    if (row_blocks == 1) {
      if (mixed || K < 2) return false;
      mixed = true;
      row_blocks = row_blocks0;
      continue;
    }
    row_blocks /= 2;
  }
  *out = g;
  return true;
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
    case LPF_E_TOO_LARGE: return "image needs more scratch than LPF_STATIC_SCRATCH_BYTES (lpf_swap_delta_static)";
    default: return "unknown error";
  }
}

extern "C" int lpf_paths_info(const lpf_paths* p, int64_t* n_half_vectors, int64_t* sum_path_len,
                              int64_t* n_trie_nodes, int* max_depth) {
  if (!p) return LPF_E_INVAL;
  if (n_half_vectors) *n_half_vectors = p->n_half;
  if (sum_path_len) *sum_path_len = p->sum_len;
  if (n_trie_nodes) *n_trie_nodes = p->n_trie_nodes;
  if (max_depth) {
    int d = 0;
    for (int o = 0; o < 4; ++o)
      for (const lpf::Node& n : p->oct[o]) d = std::max(d, (int)n.depth);
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

extern "C" int lpf_paths_program(lpf_paths* p, int H, int W, int piece_nodes, unsigned flags, uint64_t* entries,
                                 int64_t cap_entries, int64_t* n_entries, int64_t* items, int64_t cap_items,
                                 int64_t* n_items, int* n_slots, int* layout) {
  if (!p || !n_entries || !n_items || !n_slots || !layout) return LPF_E_INVAL;
  if (H < 1 || W < 1 || p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  lpf::Geom g;
  const int max_level = (flags & (LPF_NO_E2 | LPF_NO_TRIE | LPF_S2))
                            ? 0
                            : std::min(p->level_ok, p->max_level >= 0 ? p->max_level : lpf::MAX_LEVEL);
  if (!lpf::choose_geom(p->m, H, W, 1, p->max_smem > 0 ? p->max_smem : 232448, p->smem_limit, p->tile_tx, p->tile_ty,
                        p->cta_warps, max_level, lpf::max_teams_of(p), p->path_patterns, &g))
    return LPF_E_UNSUPPORTED;
  try {
    lpf::Program& pr = lpf::get_program(p, piece_nodes, flags, g.v[0].stride, g.v[1].stride, g.K, g.v[0].n_planes,
                                        g.v[0].band_words, g.v[1].band_words, g.band_rows, true);
    *n_entries = (int64_t)pr.entries.size();
    *n_items = (int64_t)pr.items.size() / 4;
    *n_slots = pr.n_slots;
    if (pr.classes.size() > LPF_LAYOUT_MAX_CLASSES) return LPF_E_UNSUPPORTED;
    for (int o = 0; o < 4; ++o) { layout[o] = pr.stride[o]; layout[4 + o] = pr.band_words[o]; }
    layout[8] = pr.K;
    layout[9] = (int)pr.classes.size();
    for (size_t c = 0; c < pr.classes.size(); ++c) {
      int* out = layout + 10 + (5 + lpf::MAX_PATTERNS) * c;
      out[0] = pr.classes[c].octant;
      out[1] = pr.classes[c].n;
      out[2] = pr.classes[c].band_words;
      out[3] = pr.classes[c].rows;
      out[4] = pr.classes[c].level;
      for (int k = 0; k < lpf::MAX_PATTERNS; ++k) out[5 + k] = k < pr.classes[c].n ? pr.classes[c].pattern[k] : -1;
    }
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
