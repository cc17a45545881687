// Host-side schedule of the V (Gram) contraction for one grid block whose packed panel has nb column
// blocks of 8 (K8 = 8 nb).  The output G = Phi^T diag(wv) Phi (LDA: upper triangle in 16-row strips;
// GGA: the full square B = Phi^T Z) is cut into passes; a pass is a band of <= 8 strips x a range of
// column blocks whose accumulators fit the registers of V_WARPS consumer warps (V_SLOTS slots of <= V_PIECE
// column blocks per warp: 15 x 2 x 4 -> 32 FP64 accumulators per lane, 128 registers per thread, 16 warps per SM;
// measured on cfg3: 8x4 5.46 ms, 11x3 4.70, 11x4 5.20, 15x3 5.06, 15x2 4.48) and whose operand columns fit one
// ring stage (<= 256).
// Inside a pass the strips are cut into pieces of <= 4 column blocks and spread over the warps by
// longest-processing-time-first, so that ragged K_p does not leave warps idle.  This is the on-device
// counterpart of the paper's pair selection + dense multiplier split.
#pragma once
#include <stdint.h>

#include <algorithm>
#include <vector>

namespace kldi {

constexpr int V_WARPS = 15, V_SLOTS = 2, V_PIECE = 4, V_BAND = 8, V_MAXCOLS = 256;
constexpr int V_ITEMS = (V_WARPS * V_SLOTS + 1) & ~1;  // VItems stored per pass (even: 16-byte bulk copies)

struct VItem {      // one slot of one consumer warp in one pass
  int32_t a;        // a_slot | b_slot << 10 | nj << 20   (stage-buffer column slots, nj = column blocks)
  int32_t b;        // arow | bcol << 16                  (packed row / column of the item's first element)
};
struct VPass {
  int32_t c1_lo, c1_n, c2_lo, c2_n;  // packed column intervals streamed into the stage (interval 2 may be empty)
  int32_t max_load, units, pad0, pad1;
};

// Exact packer of one pass: the strips' column-block widths are cut into pieces of <= V_PIECE blocks and every
// warp takes <= V_SLOTS pieces with a total load <= T.  Warps are interchangeable, so the warp being filled always
// takes its first piece from the widest remaining strip; depth-first with a waste budget (V_WARPS*T - units) and a
// node limit.  go() leaves the pieces per warp in out_s (strip index in `w`) / out_n (size, 0 = unused slot).
struct VPacker {
  int T = 0, nodes = 0;
  std::vector<int> w;  // remaining width per strip
  int out_s[V_WARPS][V_SLOTS], out_n[V_WARPS][V_SLOTS];
  bool go(int warp, int remaining) {
    static_assert(V_SLOTS == 2, "the packer fills two slots per warp");
    if (remaining == 0) {
      for (int v = warp; v < V_WARPS; ++v)
        for (int k = 0; k < V_SLOTS; ++k) out_n[v][k] = 0;
      return true;
    }
    if (warp == V_WARPS || ++nodes > 200000) return false;
    const int waste = (V_WARPS - warp) * T - remaining;
    if (waste < 0) return false;
    int big = 0;
    for (size_t i = 1; i < w.size(); ++i)
      if (w[i] > w[big]) big = (int)i;
    for (int a = std::min({V_PIECE, w[big], T}); a >= 1; --a) {
      w[big] -= a;
      out_s[warp][0] = big;
      out_n[warp][0] = a;
      for (int b = std::min(V_PIECE, T - a); b >= 0; --b) {
        if (T - a - b > waste) break;
        if (b == 0) {
          out_n[warp][1] = 0;
          if (go(warp + 1, remaining - a)) return true;
          continue;
        }
        int last = -1;
        for (size_t i = 0; i < w.size(); ++i) {
          if (w[i] < b || w[i] == last) continue;  // strips of equal remaining width are equivalent
          last = w[i];
          w[i] -= b;
          out_s[warp][1] = (int)i;
          out_n[warp][1] = b;
          if (go(warp + 1, remaining - a - b)) return true;
          w[i] += b;
        }
      }
      w[big] += a;
    }
    return false;
  }
};

// Appends the passes of an nb-block panel to `passes` (and V_WARPS*V_SLOTS items per pass to `items`).
inline void vsched_build(int nb, bool square, std::vector<VPass>& passes, std::vector<VItem>& items) {
  const int ns = (nb + 1) / 2;
  const int nbands = (ns + V_BAND - 1) / V_BAND;
  for (int band = 0; band < nbands; ++band) {
    const int s0 = (int)((int64_t)band * ns / nbands), s1 = (int)((int64_t)(band + 1) * ns / nbands);
    const int a_lo = 2 * s0, a_hi = std::min(2 * s1, nb);  // column blocks of the A rows
    int j = square ? 0 : 2 * s0;
    while (j < nb) {
      // extend [j, j1) while accumulators, slots and stage columns allow
      int j1 = j;
      for (int t = j + 1; t <= nb; ++t) {
        int units = 0, pieces = 0;
        for (int s = s0; s < s1; ++s) {
          const int lo = square ? j : std::max(j, 2 * s);
          const int w = std::max(0, t - lo);
          units += w;
          pieces += (w + V_PIECE - 1) / V_PIECE;
        }
        int cols;
        if (!square && j <= a_hi && t >= a_lo)  // one interval: union of A and B column ranges
          cols = std::max(t, a_hi) - std::min(j, a_lo);
        else
          cols = (a_hi - a_lo) + (t - j);
        if (units > V_WARPS * V_SLOTS * V_PIECE || pieces > V_WARPS * V_SLOTS || 8 * cols > V_MAXCOLS) break;
        j1 = t;
      }
      if (j1 == j) j1 = j + 1;  // cannot happen with the limits above; guards against an endless loop
      VPass P{};
      const bool one = !square && j <= a_hi && j1 >= a_lo;
      if (one) {
        P.c1_lo = 8 * std::min(j, a_lo);
        P.c1_n = 8 * (std::max(j1, a_hi) - std::min(j, a_lo));
        P.c2_lo = 0;
        P.c2_n = 0;
      } else {
        P.c1_lo = 8 * a_lo;
        P.c1_n = 8 * (a_hi - a_lo);
        P.c2_lo = 8 * j;
        P.c2_n = 8 * (j1 - j);
      }
      // pieces: try piece widths 4..1 and keep the assignment with the smallest maximum warp load
      struct Piece { int s, j0, nj; };
      const size_t item0 = items.size();
      items.resize(item0 + V_ITEMS, VItem{0, 0});
      int best_load = 1 << 30;
      for (int pw = V_PIECE; pw >= 1; --pw) {
        std::vector<Piece> pc;
        for (int s = s0; s < s1; ++s) {
          const int lo = square ? j : std::max(j, 2 * s);
          for (int c = lo; c < j1; c += pw) pc.push_back({s, c, std::min(pw, j1 - c)});
        }
        if ((int)pc.size() > V_WARPS * V_SLOTS) break;
        std::stable_sort(pc.begin(), pc.end(), [](const Piece& x, const Piece& y) { return x.nj > y.nj; });
        int load[V_WARPS] = {0}, used[V_WARPS] = {0};
        VItem trial[V_WARPS * V_SLOTS] = {};
        int units = 0;
        for (const Piece& q : pc) {
          int best = -1;
          for (int w = 0; w < V_WARPS; ++w)
            if (used[w] < V_SLOTS && (best < 0 || load[w] < load[best])) best = w;
          const int a_slot = 16 * q.s - P.c1_lo;
          const int b_slot = one ? 8 * q.j0 - P.c1_lo : P.c1_n + 8 * q.j0 - P.c2_lo;
          VItem& it = trial[best * V_SLOTS + used[best]];
          it.a = a_slot | (b_slot << 10) | (q.nj << 20);
          it.b = (16 * q.s) | ((8 * q.j0) << 16);
          load[best] += q.nj;
          used[best]++;
          units += q.nj;
        }
        const int ml = *std::max_element(load, load + V_WARPS);
        if (ml < best_load) {
          best_load = ml;
          P.max_load = ml;
          P.units = units;
          std::copy(trial, trial + V_WARPS * V_SLOTS, items.begin() + item0);
        }
      }
      // exact packer: smallest feasible maximum load below what longest-first found
      {
        std::vector<int> lo(s1 - s0), wd(s1 - s0);
        int units = 0;
        for (int s = s0; s < s1; ++s) {
          lo[s - s0] = square ? j : std::max(j, 2 * s);
          wd[s - s0] = std::max(0, j1 - lo[s - s0]);
          units += wd[s - s0];
        }
        for (int T = (units + V_WARPS - 1) / V_WARPS; T < best_load; ++T) {
          VPacker pk;
          pk.T = T;
          pk.w = wd;
          if (!pk.go(0, units)) continue;
          std::vector<int> next = lo;  // pieces of a strip are laid out left to right in warp order
          for (int w = 0; w < V_WARPS; ++w)
            for (int k = 0; k < V_SLOTS; ++k) {
              VItem it{0, 0};
              const int nj = pk.out_n[w][k];
              if (nj) {
                const int s = s0 + pk.out_s[w][k], j0 = next[pk.out_s[w][k]];
                next[pk.out_s[w][k]] += nj;
                const int a_slot = 16 * s - P.c1_lo;
                const int b_slot = one ? 8 * j0 - P.c1_lo : P.c1_n + 8 * j0 - P.c2_lo;
                it.a = a_slot | (b_slot << 10) | (nj << 20);
                it.b = (16 * s) | ((8 * j0) << 16);
              }
              items[item0 + w * V_SLOTS + k] = it;
            }
          best_load = T;
          P.max_load = T;
          P.units = units;
          break;
        }
      }
      passes.push_back(P);
      j = j1;
    }
  }
}

}  // namespace kldi
