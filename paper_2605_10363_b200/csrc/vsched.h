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
  int32_t a;        // a_slot | b_slot << 10 | nj << 20 | diag << 24  (stage-buffer column slots, nj = column blocks,
                    // diag: the item starts on the diagonal, rows 8..15 of its first block are not computed)
  int32_t b;        // arow | bcol << 16                  (packed row / column of the item's first element)
};
struct VPass {
  int32_t c1_lo, c1_n, c2_lo, c2_n;  // packed column intervals streamed into the stage (interval 2 may be empty)
  int32_t max_load, units, smsp_load, pad1;  // max load of a warp / of a scheduler partition (warps w % 4) and the
                                             // pass total, in 8x8 blocks (one DMMA per k-step each)
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
      // Pieces -> warps.  The FP64 tensor pipe belongs to a scheduler partition (SMSP = warp % 4), and 15 consumer
      // warps leave partition 3 with three of them (the producer is the fourth), so the quantity to balance is the
      // load per partition, not per warp: pieces are spread longest-first over the four partitions (slot limits
      // 2 x warps of the partition), then pieces of the fullest partition are moved or split towards the emptiest
      // while that lowers the maximum, and each partition deals its pieces to its own warps.
      // cost of a piece in 8x8 blocks (= DMMAs per k-step): 2 per column block, minus the lower 8 rows of the strip's
      // first block on the diagonal, which lie strictly below it and are not computed (VItem diag flag)
      struct Piece {
        int s, j0, nj, diag;
        int cost() const { return 2 * nj - diag; }
      };
      const size_t item0 = items.size();
      items.resize(item0 + V_ITEMS, VItem{0, 0});
      int nwq[4] = {0, 0, 0, 0};
      for (int w = 0; w < V_WARPS; ++w) nwq[w & 3]++;
      int best_q = 1 << 30, best_w = 1 << 30;
      for (int pw = V_PIECE; pw >= 1; --pw) {
        std::vector<Piece> pc;
        for (int s = s0; s < s1; ++s) {
          const int lo = square ? j : std::max(j, 2 * s);
          for (int c = lo; c < j1; c += pw) pc.push_back({s, c, std::min(pw, j1 - c), (!square && c == 2 * s) ? 1 : 0});
        }
        if ((int)pc.size() > V_WARPS * V_SLOTS) break;
        std::stable_sort(pc.begin(), pc.end(), [](const Piece& x, const Piece& y) { return x.cost() > y.cost(); });
        std::vector<Piece> bin[4];
        int load[4] = {0, 0, 0, 0};
        bool ok = true;
        for (const Piece& q : pc) {
          int best = -1;
          for (int b = 0; b < 4; ++b)
            if ((int)bin[b].size() < V_SLOTS * nwq[b] && (best < 0 || load[b] < load[best])) best = b;
          if (best < 0) { ok = false; break; }
          bin[best].push_back(q);
          load[best] += q.cost();
        }
        if (!ok) continue;
        for (int iter = 0; iter < 64; ++iter) {  // move / split from the fullest to the emptiest partition
          int hi = 0, lo = 0;
          for (int b = 1; b < 4; ++b) {
            if (load[b] > load[hi]) hi = b;
            if (load[b] < load[lo]) lo = b;
          }
          const int gap = load[hi] - load[lo];
          if (gap < 2 || (int)bin[lo].size() >= V_SLOTS * nwq[lo]) break;
          const int want = gap / 2;  // in 8x8 blocks
          int pick = -1;  // largest piece not larger than want, else any piece to split
          for (size_t i = 0; i < bin[hi].size(); ++i)
            if (bin[hi][i].cost() <= want && (pick < 0 || bin[hi][i].cost() > bin[hi][pick].cost())) pick = (int)i;
          if (pick >= 0) {
            bin[lo].push_back(bin[hi][pick]);
            load[lo] += bin[hi][pick].cost();
            load[hi] -= bin[hi][pick].cost();
            bin[hi].erase(bin[hi].begin() + pick);
            continue;
          }
          const int cut = want / 2;  // whole column blocks split off the tail of a piece (the diag flag stays in front)
          if (cut < 1) break;
          for (size_t i = 0; i < bin[hi].size(); ++i)
            if (bin[hi][i].nj > cut) { pick = (int)i; break; }
          if (pick < 0) break;
          Piece& src = bin[hi][pick];
          src.nj -= cut;
          bin[lo].push_back({src.s, src.j0 + src.nj, cut, 0});
          load[hi] -= 2 * cut;
          load[lo] += 2 * cut;
        }
        const int mq = *std::max_element(load, load + 4);
        // deal the pieces of a partition to its warps: largest first, then back in reverse order
        VItem trial[V_WARPS * V_SLOTS] = {};
        int wload[V_WARPS] = {0};
        int units = 0;
        for (int b = 0; b < 4; ++b) {
          std::stable_sort(bin[b].begin(), bin[b].end(), [](const Piece& x, const Piece& y) { return x.cost() > y.cost(); });
          int used[(V_WARPS + 3) / 4] = {0};
          for (const Piece& q : bin[b]) {
            int bw = -1;
            for (int i = 0; i < nwq[b]; ++i)
              if (used[i] < V_SLOTS && (bw < 0 || wload[b + 4 * i] < wload[b + 4 * bw])) bw = i;
            const int w = b + 4 * bw;
            const int a_slot = 16 * q.s - P.c1_lo;
            const int b_slot = one ? 8 * q.j0 - P.c1_lo : P.c1_n + 8 * q.j0 - P.c2_lo;
            VItem& it = trial[w * V_SLOTS + used[bw]];
            it.a = a_slot | (b_slot << 10) | (q.nj << 20) | (q.diag << 24);
            it.b = (16 * q.s) | ((8 * q.j0) << 16);
            wload[w] += q.cost();
            used[bw]++;
            units += q.cost();
          }
        }
        const int mw = *std::max_element(wload, wload + V_WARPS);
        if (mq < best_q || (mq == best_q && mw < best_w)) {
          best_q = mq;
          best_w = mw;
          P.max_load = mw;
          P.smsp_load = mq;
          P.units = units;
          std::copy(trial, trial + V_WARPS * V_SLOTS, items.begin() + item0);
        }
      }
      passes.push_back(P);
      j = j1;
    }
  }
}

}  // namespace kldi
