// chol_schedule.cu -- host side of rows c, d1: the static schedule of the tile task
// graph that `chol_task_kernel` (cholesky.cu) executes.
//
// Tiles are 64x64; nt = ceil(p/64).  Task graph (left-looking, see cholesky.cu for the algebra):
//   L(i,j), i >= j : acc = Q_ij - sum_{k<j} L_ik L_jk^T ;  i == j: potrf + inverse of the diagonal tile ;
//                                                          i >  j: L_ij = acc W_jj^T
//   B(i,j), i <  j : acc = - sum_{k=i}^{j-1} L_jk Wt_ik^T ; W_ji = W_jj acc      (same inverse super-block only)
// A k-loop only needs FRESH data in its last step, so the tiles on the critical path -- the diagonal and
// the first sub-diagonal of every column -- are split into a prefix task (stores the partial accumulator to a
// workspace slot) and a short finish.  With K >= 2 CTAs the finishes are the CHAIN tasks of the first list (a
// dedicated CTA, operands kept in its shared memory): POTRF(j) (type 2: potrf + inverse of the diagonal tile),
// TRSM(j) (type 3: L(j+1,j) from the parked accumulator with every k < j applied) and SYRK(j) (type 4: the last
// update of A(j+1,j+1)); with K = 1 they are ordinary finish tasks of type 0.  Every CTA runs its own list in order and
// waits on per-tile flags inside a task; the lists are subsequences of one global order in which every
// producer is placed before its consumers, so with all CTAs co-resident the spin-waits cannot deadlock.
// The lists come from a greedy list scheduler driven by a cost model of the kernel (microseconds below,
// measured on B200), which also gives the makespan estimate the orchestrator uses to size the SM split.
#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <queue>
#include <vector>
#include "hsp_internal.h"

namespace hsp {

namespace {

// us, from the chol_trace option at p = 1000 and p = 4000 (profiles/r02_c_cholesky.md).  mac: one 64x64x64 product of a k-loop (TMA-fed,
// DMMA peak 2.08); fin: finish of an off-diagonal tile (wait for W_jj, load it, product, store, flag); cmac: a product of the
// chain CTA, operands in shared memory; cpub: W_jj reaches global memory (publisher warp) that long after the inverse
struct Cost { double mac = 2.4, hop = 2.0, potrf = 7.9, trinv = 1.9, store = 0.9, loadp = 0.3, cmac = 2.6, fin = 4.7, cpub = 0.5; };

struct Step { double cost; int dep[2]; bool local = false; };   // deps are task ids (-1 = none); local: dep[0] ran on the same CTA (no flag hop)
struct Node {
  CholTask t;
  std::vector<Step> steps;
  std::vector<int> prod;                                  // distinct producers
  std::vector<std::pair<int, int>> cons;                  // (consumer task, step index)
  double total = 0.0, rank = 0.0;
};

struct Graph {
  std::vector<Node> n;
  std::vector<int> chain;                                  // ids of the chain tasks, in execution order
  int n_slots = 0;
};

Graph build_graph(int nt, int sb, const Cost& c, bool chain) {
  Graph g;
  std::vector<int> idL((size_t)nt * nt, -1), idB((size_t)nt * nt, -1);
  auto add = [&](const CholTask& t) { g.n.push_back(Node{t, {}, {}, {}, 0.0, 0.0}); return (int)g.n.size() - 1; };
  // L tiles, column by column (ids increase along a valid topological order)
  if (chain) {
    int prev = -1;                                         // previous chain task (same CTA: runs in order)
    for (int j = 0; j < nt; ++j) {
      // prefix of the sub-diagonal tile (j+1, j): every k < j;  prefix of the NEXT diagonal tile (j+1, j+1): every k < j
      int ps = -1, pd = -1, slot_s = -1, slot_d = -1;
      if (j + 1 < nt && j >= 1) {
        slot_s = g.n_slots++;
        ps = add(CholTask{0, j + 1, j, 0, j, -1, slot_s, 0});
        for (int k = 0; k < j; ++k) g.n[ps].steps.push_back(Step{c.mac, {idL[(size_t)(j + 1) * nt + k], idL[(size_t)j * nt + k]}});
        g.n[ps].steps.push_back(Step{c.store, {-1, -1}});
        slot_d = g.n_slots++;
        pd = add(CholTask{0, j + 1, j + 1, 0, j, -1, slot_d, 0});
        for (int k = 0; k < j; ++k) g.n[pd].steps.push_back(Step{c.mac, {idL[(size_t)(j + 1) * nt + k], -1}});
        g.n[pd].steps.push_back(Step{c.store, {-1, -1}});
      }
      const int po = add(CholTask{2, j, j, 0, 0, -1, -1, 0});
      g.n[po].steps.push_back(Step{c.potrf + c.trinv + c.cpub, {prev, -1}, true});
      g.chain.push_back(po); prev = po;
      idL[(size_t)j * nt + j] = po;
      if (j + 1 < nt) {
        const int tr = add(CholTask{3, j + 1, j, 0, 0, slot_s, -1, 0});
        g.n[tr].steps.push_back(Step{c.loadp + c.cmac + c.store - c.cpub, {po, ps}, true});
        g.chain.push_back(tr);
        idL[(size_t)(j + 1) * nt + j] = tr;
        const int sy = add(CholTask{4, j + 1, j, 0, 0, slot_d, -1, 0});
        g.n[sy].steps.push_back(Step{c.loadp + c.cmac, {tr, pd}, true});
        g.chain.push_back(sy); prev = sy;
      }
      for (int i = j + 2; i < nt; ++i) {
        const int id = add(CholTask{0, i, j, 0, j, -1, -1, 0});
        for (int k = 0; k < j; ++k) g.n[id].steps.push_back(Step{c.mac, {idL[(size_t)i * nt + k], idL[(size_t)j * nt + k]}});
        g.n[id].steps.push_back(Step{c.fin, {po, -1}});
        idL[(size_t)i * nt + j] = id;
      }
    }
  } else
  for (int j = 0; j < nt; ++j)
    for (int i = j; i < nt; ++i) {
      const bool split = (i == j || i == j + 1) && j >= 2;
      int k0 = 0, pre = -1, slot = -1;
      if (split) {
        slot = g.n_slots++;
        pre = add(CholTask{0, i, j, 0, j - 1, -1, slot, 0});
        for (int k = 0; k < j - 1; ++k) g.n[pre].steps.push_back(Step{c.mac, {idL[(size_t)i * nt + k], i != j ? idL[(size_t)j * nt + k] : -1}});
        g.n[pre].steps.push_back(Step{c.store, {-1, -1}});
        k0 = j - 1;
      }
      const int id = add(CholTask{0, i, j, k0, j, slot, -1, 0});
      if (split) g.n[id].steps.push_back(Step{c.loadp, {pre, -1}});
      for (int k = k0; k < j; ++k) g.n[id].steps.push_back(Step{c.mac, {idL[(size_t)i * nt + k], i != j ? idL[(size_t)j * nt + k] : -1}});
      if (i == j) g.n[id].steps.push_back(Step{c.potrf + c.trinv + c.store, {-1, -1}});
      else g.n[id].steps.push_back(Step{c.fin, {idL[(size_t)j * nt + j], -1}});
      idL[(size_t)i * nt + j] = id;
    }
  // inverse tiles W(j,i), i < j, inside one super-block of sb tiles
  for (int j = 0; j < nt; ++j)
    for (int i = 0; i < j; ++i) {
      if (i / sb != j / sb) continue;
      const int id = add(CholTask{1, i, j, i, j, -1, -1, 0});
      for (int k = i; k < j; ++k)
        g.n[id].steps.push_back(Step{c.mac, {idL[(size_t)j * nt + k], k == i ? idL[(size_t)i * nt + i] : idB[(size_t)i * nt + k]}});
      g.n[id].steps.push_back(Step{c.fin, {idL[(size_t)j * nt + j], -1}});
      idB[(size_t)i * nt + j] = id;
    }
  for (size_t a = 0; a < g.n.size(); ++a) {
    Node& nd = g.n[a];
    for (size_t s = 0; s < nd.steps.size(); ++s) {
      nd.total += nd.steps[s].cost;
      for (int d : nd.steps[s].dep)
        if (d >= 0) {
          if (std::find(nd.prod.begin(), nd.prod.end(), d) == nd.prod.end()) nd.prod.push_back(d);
          g.n[d].cons.push_back({(int)a, (int)s});
        }
    }
  }
  // upward rank: time from the start of a task to the end of the graph with unlimited CTAs.
  // ids are topologically ordered except that B tiles depend on L tiles of any column: process in
  // reverse order of a topological sort.
  std::vector<int> order, indeg(g.n.size());
  for (size_t a = 0; a < g.n.size(); ++a) indeg[a] = (int)g.n[a].prod.size();
  std::vector<int> stack;
  for (size_t a = 0; a < g.n.size(); ++a) if (!indeg[a]) stack.push_back((int)a);
  std::vector<std::vector<int>> succ(g.n.size());
  for (size_t a = 0; a < g.n.size(); ++a) for (int d : g.n[a].prod) succ[d].push_back((int)a);
  while (!stack.empty()) {
    const int a = stack.back(); stack.pop_back(); order.push_back(a);
    for (int s : succ[a]) if (--indeg[s] == 0) stack.push_back(s);
  }
  std::vector<double> after(g.n.size(), 0.0);
  for (auto it = order.rbegin(); it != order.rend(); ++it) {
    Node& nd = g.n[*it];
    double best = 0.0;
    for (auto& cs : nd.cons) {
      const Node& cn = g.n[cs.first];
      double rem = 0.0;
      for (size_t s = cs.second; s < cn.steps.size(); ++s) rem += cn.steps[s].cost;
      best = std::max(best, c.hop + rem + after[cs.first]);
    }
    after[*it] = best;
    nd.rank = nd.total + best;
  }
  return g;
}

// Execute task `nd` from time `start` with the known finish times of its producers.
inline void run_task(const Node& nd, double start, const std::vector<double>& finish, double hop, double* end, double* idle) {
  double cur = start, id = 0.0;
  for (const Step& s : nd.steps) {
    double r = 0.0;
    for (int q = 0; q < 2; ++q) if (s.dep[q] >= 0) r = std::max(r, finish[s.dep[q]] + (q == 0 && s.local ? 0.0 : hop));
    if (r > cur) { id += r - cur; cur = r; }
    cur += s.cost;
  }
  *end = cur; *idle = id;
}

}  // namespace

CholSchedule chol_build_schedule(int nt, int sb, int K) {
  const Cost c;
  const bool big = nt > 96;                              // the greedy search is quadratic in the task count
  const bool chain = K >= 2 && nt >= 2 && !big;          // list 0 = the chain CTA, lists 1.. = everything else
  Graph g = build_graph(nt, sb, c, chain);
  const int T = (int)g.n.size();
  CholSchedule out;
  out.K = K; out.n_slots = g.n_slots;
  std::vector<std::vector<int>> lists(K);
  std::vector<double> finish(T, 0.0);
  if (big || K == 1) {
    // deal the tasks round-robin in id order (a valid global order: every producer has a smaller id or is an
    // L tile of an earlier column)
    std::vector<int> order(T);
    for (int a = 0; a < T; ++a) order[a] = a;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
      const CholTask &x = g.n[a].t, &y = g.n[b].t;
      if (x.j != y.j) return x.j < y.j;
      return x.type < y.type;
    });
    std::vector<double> free_at(K, 0.0);
    int q = 0;
    for (int a : order) {
      const int cta = q++ % K;
      double e, idle;
      run_task(g.n[a], free_at[cta], finish, c.hop, &e, &idle);
      finish[a] = e; free_at[cta] = e;
      lists[cta].push_back(a);
    }
  } else {
    std::vector<char> in_cand(T, 0), placed_v(T, 0), is_chain(T, 0);
    for (int a : g.chain) is_chain[a] = 1;
    std::vector<int> cand;
    int placed = 0;
    size_t chain_pos = 0;
    double chain_free = 0.0;
    auto ready = [&](int a) {
      for (int d : g.n[a].prod) if (!placed_v[d]) return false;
      return true;
    };
    auto release = [&](int a) {                            // consumers of a placed task become candidates
      for (auto& cs : g.n[a].cons)
        if (!in_cand[cs.first] && !is_chain[cs.first] && ready(cs.first)) { cand.push_back(cs.first); in_cand[cs.first] = 1; }
    };
    // the chain CTA takes its next task as soon as all its producers are placed (placement order = the global order)
    auto advance_chain = [&]() {
      while (chain_pos < g.chain.size() && ready(g.chain[chain_pos])) {
        const int a = g.chain[chain_pos++];
        double e, idle;
        run_task(g.n[a], chain_free, finish, c.hop, &e, &idle);
        finish[a] = e; chain_free = e; placed_v[a] = 1; ++placed;
        lists[0].push_back(a);
        release(a);
      }
    };
    for (int a = 0; a < T; ++a) if (!is_chain[a] && g.n[a].prod.empty()) { cand.push_back(a); in_cand[a] = 1; }
    using Ev = std::pair<double, int>;
    std::priority_queue<Ev, std::vector<Ev>, std::greater<Ev>> free_q;
    for (int k = chain ? 1 : 0; k < K; ++k) free_q.push({0.0, k});
    const double idle_ok = 1.0;
    advance_chain();
    while (placed < T) {
      if (cand.empty()) { fprintf(stderr, "chol_build_schedule: no candidate (nt=%d K=%d)\n", nt, K); abort(); }
      const Ev ev = free_q.top(); free_q.pop();
      int best = -1; double best_end = 0.0, best_rank = -1.0;
      int fb = -1; double fb_end = 0.0, fb_idle = 1e300, fb_rank = -1.0;
      for (int a : cand) {
        double e, idle;
        run_task(g.n[a], ev.first, finish, c.hop, &e, &idle);
        if (idle <= idle_ok) {
          if (g.n[a].rank > best_rank) { best = a; best_end = e; best_rank = g.n[a].rank; }
        } else if (idle < fb_idle || (idle == fb_idle && g.n[a].rank > fb_rank)) {
          fb = a; fb_end = e; fb_idle = idle; fb_rank = g.n[a].rank;
        }
      }
      const int a = best >= 0 ? best : fb;
      const double e = best >= 0 ? best_end : fb_end;
      cand.erase(std::find(cand.begin(), cand.end(), a));
      finish[a] = e; placed_v[a] = 1; ++placed;
      lists[ev.second].push_back(a);
      free_q.push({e, ev.second});
      release(a);
      advance_chain();
    }
  }
  out.list_off.assign(K + 1, 0);
  for (int k = 0; k < K; ++k) {
    out.list_off[k + 1] = out.list_off[k] + (int)lists[k].size();
    for (int a : lists[k]) out.tasks.push_back(g.n[a].t);
  }
  out.makespan_us = 0.0;
  for (int a = 0; a < T; ++a) out.makespan_us = std::max(out.makespan_us, finish[a]);
  return out;
}

}  // namespace hsp
