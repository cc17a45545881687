// P2 alternative: overlap-signature ordering of the AO blocks (Eq. 8-10,
// PAPER.md:444-457 Eq. 21).  Host code, once per geometry.
//
// The paper orders basis functions by clustering the rows of the overlap matrix S (Eq. 8): signature s_i = row i of S
// (Eq. 9), cosine distance d(i,j) = 1 - s_i.s_j / (|s_i||s_j|) (Eq. 21), agglomerative clustering with average
// linkage, sub-trees oriented at each merge so that their closest leaves are adjacent, leaf order = permutation.
// Here the clustered unit is the CENTRE (reading A16): the block filter and the panel packing act per
// shell, shells of one centre have (nearly) the same signature, and the order only decides where an atom's AO blocks
// sit in D and V, so the signature of atom A is the row (T_A1 .. T_AN) of the atom-block overlap norms
// T_AB = || S_AB ||_F, computed in closed form (Obara-Saika recursion for Cartesian Gaussians, l <= 2).
#include <algorithm>
#include <cmath>
#include <numeric>
#include <vector>

#include "kldi_internal.h"

namespace kldi {

namespace {
// 1-D overlap integrals s[i][j] = int (x-A)^i (x-B)^j exp(-a (x-A)^2 - b (x-B)^2) dx, i, j <= 2 (Obara-Saika)
void overlap_1d(double a, double b, double A, double B, double (&s)[3][3]) {
  const double p = a + b, mu = a * b / p, P = (a * A + b * B) / p, XPA = P - A, XPB = P - B, h = 0.5 / p;
  s[0][0] = std::sqrt(M_PI / p) * std::exp(-mu * (A - B) * (A - B));
  for (int j = 0; j < 3; ++j) {
    if (j > 0) s[0][j] = XPB * s[0][j - 1] + (j > 1 ? h * (j - 1) * s[0][j - 2] : 0.0);
    for (int i = 1; i < 3; ++i)
      s[i][j] = XPA * s[i - 1][j] + h * ((i > 1 ? (i - 1) * s[i - 2][j] : 0.0) + (j > 0 ? j * s[i - 1][j - 1] : 0.0));
  }
}
double dfact(int n) {
  double r = 1.0;
  for (; n > 1; n -= 2) r *= n;
  return r;
}
const int CART[3][6][3] = {{{0, 0, 0}},
                           {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}},
                           {{2, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}}};
}  // namespace

// sum over the Cartesian components and primitives of two shells of S_ij^2 (squared Frobenius norm of the block)
static double shell_pair_norm2(const kldi_shells* sh, int sa, int sb, const double* A, const double* B) {
  const int la = sh->l[sa], lb = sh->l[sb], na = (la + 1) * (la + 2) / 2, nb = (lb + 1) * (lb + 2) / 2;
  double blk[6][6] = {};
  for (int pa = sh->nprim_off[sa]; pa < sh->nprim_off[sa + 1]; ++pa)
    for (int pb = sh->nprim_off[sb]; pb < sh->nprim_off[sb + 1]; ++pb) {
      const double a = sh->alpha[pa], b = sh->alpha[pb];
      double s1[3][3][3];
      for (int d = 0; d < 3; ++d) overlap_1d(a, b, A[d], B[d], s1[d]);
      const double ca = sh->coef[pa] * std::pow(2.0 * a / M_PI, 0.75) * std::pow(4.0 * a, 0.5 * la);
      const double cb = sh->coef[pb] * std::pow(2.0 * b / M_PI, 0.75) * std::pow(4.0 * b, 0.5 * lb);
      for (int i = 0; i < na; ++i)
        for (int j = 0; j < nb; ++j) {
          const int* u = CART[la][i];
          const int* v = CART[lb][j];
          const double ni = 1.0 / std::sqrt(dfact(2 * u[0] - 1) * dfact(2 * u[1] - 1) * dfact(2 * u[2] - 1));
          const double nj = 1.0 / std::sqrt(dfact(2 * v[0] - 1) * dfact(2 * v[1] - 1) * dfact(2 * v[2] - 1));
          blk[i][j] += ca * cb * ni * nj * s1[0][u[0]][v[0]] * s1[1][u[1]][v[1]] * s1[2][u[2]][v[2]];
        }
    }
  double t = 0.0;
  for (int i = 0; i < na; ++i)
    for (int j = 0; j < nb; ++j) t += blk[i][j] * blk[i][j];
  return t;
}

// Atom order by overlap-signature clustering.  Returns false (order untouched) when the input is outside what this
// host implementation handles (more than 4096 centres: the distance matrix is O(N^2)).
bool overlap_signature_order(const kldi_atoms* atoms, const kldi_shells* shells, std::vector<int>& order,
                             std::vector<double>* dist_out) {
  const int n = atoms->n_atoms;
  if (n > 4096) return false;
  order.resize(n);
  std::iota(order.begin(), order.end(), 0);
  if (n < 3) return true;
  std::vector<std::vector<int>> sh_of(n);
  for (int s = 0; s < shells->n_shells; ++s) sh_of[shells->atom[s]].push_back(s);
  // T_AB = ||S_AB||_F (Eq. 8 on atom blocks)
  std::vector<double> T((size_t)n * n, 0.0);
  for (int a = 0; a < n; ++a)
    for (int b = a; b < n; ++b) {
      double t = 0.0;
      for (int sa : sh_of[a])
        for (int sb : sh_of[b]) t += shell_pair_norm2(shells, sa, sb, atoms->xyz + 3 * a, atoms->xyz + 3 * b);
      T[(size_t)a * n + b] = T[(size_t)b * n + a] = std::sqrt(t);
    }
  // cosine distance of the signatures (Eq. 9, 10, 21)
  std::vector<double> nrm(n, 0.0);
  for (int a = 0; a < n; ++a) {
    double t = 0.0;
    for (int c = 0; c < n; ++c) t += T[(size_t)a * n + c] * T[(size_t)a * n + c];
    nrm[a] = std::sqrt(t);
  }
  std::vector<double> d((size_t)n * n, 0.0);
  for (int a = 0; a < n; ++a)
    for (int b = a + 1; b < n; ++b) {
      double dot = 0.0;
      for (int c = 0; c < n; ++c) dot += T[(size_t)a * n + c] * T[(size_t)b * n + c];
      const double v = (nrm[a] > 0 && nrm[b] > 0) ? 1.0 - dot / (nrm[a] * nrm[b]) : 1.0;
      d[(size_t)a * n + b] = d[(size_t)b * n + a] = v < 0 ? 0.0 : v;
    }
  if (dist_out) *dist_out = d;
  // average-linkage agglomeration (Lance-Williams update of the cluster distance matrix D), leaf lists oriented at
  // every merge so that the closest of the four end-leaf pairs becomes adjacent (reading A16)
  std::vector<double> D = d;
  std::vector<std::vector<int>> leaves(n);
  std::vector<int> size(n, 1), nn(n, -1);
  std::vector<char> alive(n, 1);
  for (int a = 0; a < n; ++a) leaves[a] = {a};
  auto find_nn = [&](int a) {
    int best = -1;
    for (int b = 0; b < n; ++b)
      if (b != a && alive[b] && (best < 0 || D[(size_t)a * n + b] < D[(size_t)a * n + best])) best = b;
    nn[a] = best;
  };
  for (int a = 0; a < n; ++a) find_nn(a);
  for (int step = 0; step < n - 1; ++step) {
    int x = -1;
    for (int a = 0; a < n; ++a)
      if (alive[a] && (x < 0 || D[(size_t)a * n + nn[a]] < D[(size_t)x * n + nn[x]])) x = a;
    int y = nn[x];
    if (y < x) std::swap(x, y);
    // orientation: ends (x first/last) x (y first/last)
    std::vector<int>&lx = leaves[x], &ly = leaves[y];
    const double c_ll = d[(size_t)lx.back() * n + ly.front()], c_lr = d[(size_t)lx.back() * n + ly.back()];
    const double c_fl = d[(size_t)lx.front() * n + ly.front()], c_fr = d[(size_t)lx.front() * n + ly.back()];
    const double best = std::min(std::min(c_ll, c_lr), std::min(c_fl, c_fr));
    if (best == c_ll) {
    } else if (best == c_lr) {
      std::reverse(ly.begin(), ly.end());
    } else if (best == c_fl) {
      std::reverse(lx.begin(), lx.end());
    } else {
      std::reverse(lx.begin(), lx.end());
      std::reverse(ly.begin(), ly.end());
    }
    lx.insert(lx.end(), ly.begin(), ly.end());
    ly.clear();
    // average linkage: D(x u y, z) = (|x| D(x,z) + |y| D(y,z)) / (|x| + |y|)
    for (int z = 0; z < n; ++z)
      if (alive[z] && z != x && z != y) {
        const double v = (size[x] * D[(size_t)x * n + z] + size[y] * D[(size_t)y * n + z]) / (size[x] + size[y]);
        D[(size_t)x * n + z] = D[(size_t)z * n + x] = v;
      }
    size[x] += size[y];
    alive[y] = 0;
    find_nn(x);
    for (int z = 0; z < n; ++z)
      if (alive[z] && z != x) {
        if (nn[z] == x || nn[z] == y) find_nn(z);
        else if (D[(size_t)z * n + x] < D[(size_t)z * n + nn[z]]) nn[z] = x;
      }
  }
  for (int a = 0; a < n; ++a)
    if (alive[a]) order = leaves[a];
  return (int)order.size() == n;
}

}  // namespace kldi
