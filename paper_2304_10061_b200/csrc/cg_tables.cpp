// Host-side construction of the tensor-track tables: irreps per layer, paths, real Clebsch-Gordan
// blocks, and the path-weight-fused sparse tensor K^L (Fig. 3 PAPER.md:180;
// conventions SURVEY.md §8(c) S5/S6).  Independent of oracle/ (no shared code).
#include <algorithm>
#include <cmath>
#include <complex>
#include <map>
#include <set>

#include "internal.h"

namespace {

double fact(int n) {
  double r = 1.0;
  for (int k = 2; k <= n; ++k) r *= k;
  return r;
}

// <j1 m1 j2 m2 | j m>, Condon-Shortley phase, Racah's closed form.
double clebsch(int j1, int m1, int j2, int m2, int j, int m) {
  if (m1 + m2 != m || j < std::abs(j1 - j2) || j > j1 + j2) return 0.0;
  if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(m) > j) return 0.0;
  double delta = fact(j1 + j2 - j) * fact(j1 - j2 + j) * fact(-j1 + j2 + j) / fact(j1 + j2 + j + 1);
  double pre = (2 * j + 1) * delta * fact(j + m) * fact(j - m) * fact(j1 + m1) * fact(j1 - m1) * fact(j2 + m2) *
               fact(j2 - m2);
  double sum = 0.0;
  for (int k = 0; k <= j1 + j2 - j; ++k) {
    int t1 = j1 + j2 - j - k, t2 = j1 - m1 - k, t3 = j2 + m2 - k, t4 = j - j2 + m1 + k, t5 = j - j1 - m2 + k;
    if (t1 < 0 || t2 < 0 || t3 < 0 || t4 < 0 || t5 < 0) continue;
    double den = fact(k) * fact(t1) * fact(t2) * fact(t3) * fact(t4) * fact(t5);
    sum += ((k & 1) ? -1.0 : 1.0) / den;
  }
  return std::sqrt(pre) * sum;
}

typedef std::complex<double> cd;

// Unitary change of basis complex -> real harmonics, rows = real index (m_r + l), cols = complex m + l.
// m_r > 0: ((-1)^m Y_m + Y_-m)/sqrt2 ; m_r = 0: Y_0 ; m_r < 0: i (Y_-|m| - (-1)^m Y_|m|)/sqrt2.
std::vector<cd> real_from_complex(int l) {
  int n = 2 * l + 1;
  std::vector<cd> U(n * n, cd(0, 0));
  const double s = 1.0 / std::sqrt(2.0);
  U[l * n + l] = 1.0;
  for (int m = 1; m <= l; ++m) {
    double sg = (m & 1) ? -1.0 : 1.0;
    U[(l + m) * n + (l + m)] = sg * s;
    U[(l + m) * n + (l - m)] = s;
    U[(l - m) * n + (l - m)] = cd(0, s);
    U[(l - m) * n + (l + m)] = cd(0, -sg * s);
  }
  return U;
}

// Real CG block C[a][b][c]; components of real tensors x_r = U x_c, hence
// C = sum conj(U1[a,m1]) conj(U2[b,m2]) Uo[c,mo] <l1 m1 l2 m2|lo mo>, purely real or purely imaginary.
std::vector<double> real_cg_block(int l1, int l2, int lo) {
  int n1 = 2 * l1 + 1, n2 = 2 * l2 + 1, no = 2 * lo + 1;
  std::vector<cd> U1 = real_from_complex(l1), U2 = real_from_complex(l2), Uo = real_from_complex(lo);
  std::vector<cd> C(n1 * n2 * no, cd(0, 0));
  for (int m1 = -l1; m1 <= l1; ++m1)
    for (int m2 = -l2; m2 <= l2; ++m2) {
      int mo = m1 + m2;
      if (std::abs(mo) > lo) continue;
      double g = clebsch(l1, m1, l2, m2, lo, mo);
      if (g == 0.0) continue;
      for (int a = 0; a < n1; ++a) {
        cd u1 = std::conj(U1[a * n1 + (m1 + l1)]);
        if (u1 == cd(0, 0)) continue;
        for (int b = 0; b < n2; ++b) {
          cd u2 = std::conj(U2[b * n2 + (m2 + l2)]);
          if (u2 == cd(0, 0)) continue;
          for (int c = 0; c < no; ++c) C[(a * n2 + b) * no + c] += u1 * u2 * Uo[c * no + (mo + lo)] * g;
        }
      }
    }
  std::vector<double> R(n1 * n2 * no);
  bool even = ((l1 + l2 + lo) % 2) == 0;
  for (size_t k = 0; k < C.size(); ++k) R[k] = even ? C[k].real() : C[k].imag();
  // sign rule: first entry (a,b,c lexicographic) with |v| > 1e-12 is positive
  for (size_t k = 0; k < R.size(); ++k)
    if (std::fabs(R[k]) > 1e-12) {
      if (R[k] < 0)
        for (auto& v : R) v = -v;
      break;
    }
  for (auto& v : R)
    if (std::fabs(v) < 1e-14) v = 0.0;
  return R;
}

bool natural(const Irrep& ir) { return ir.p == ((ir.l & 1) ? -1 : 1); }

void sort_irreps(std::vector<Irrep>& v) {
  std::sort(v.begin(), v.end(), [](const Irrep& a, const Irrep& b) {
    if (a.l != b.l) return a.l < b.l;
    return (natural(a) ? 0 : 1) < (natural(b) ? 0 : 1);
  });
  v.erase(std::unique(v.begin(), v.end(), [](const Irrep& a, const Irrep& b) { return a.l == b.l && a.p == b.p; }),
          v.end());
}

}  // namespace

void al_enumerate(int lmax, int NL, std::vector<std::vector<Irrep>>& S,
                  std::vector<std::vector<TPLayerHost::Path>>& paths) {
  std::vector<Irrep> env;
  for (int l = 0; l <= lmax; ++l) env.push_back({l, (l & 1) ? -1 : 1});
  // forward reachability
  std::vector<std::vector<Irrep>> O(NL + 1);
  O[0] = env;
  for (int L = 1; L <= NL; ++L) {
    std::vector<Irrep> nxt;
    for (auto& i1 : O[L - 1])
      for (auto& i2 : env)
        for (int lo = std::abs(i1.l - i2.l); lo <= std::min(i1.l + i2.l, lmax); ++lo) nxt.push_back({lo, i1.p * i2.p});
    sort_irreps(nxt);
    O[L] = nxt;
  }
  // backward pruning: keep what can still reach the final scalars
  S.assign(NL + 1, {});
  S[NL] = {Irrep{0, 1}};
  for (int L = NL - 1; L >= 0; --L) {
    for (auto& i1 : O[L]) {
      bool ok = false;
      for (auto& i2 : env)
        for (auto& io : S[L + 1])
          if (std::abs(i1.l - i2.l) <= io.l && io.l <= i1.l + i2.l && io.p == i1.p * i2.p) ok = true;
      if (ok) S[L].push_back(i1);
    }
    sort_irreps(S[L]);
  }
  paths.assign(NL, {});
  for (int L = 1; L <= NL; ++L)
    for (int i1 = 0; i1 < (int)S[L - 1].size(); ++i1)
      for (int l2 = 0; l2 <= lmax; ++l2)
        for (int io = 0; io < (int)S[L].size(); ++io) {
          const Irrep &a = S[L - 1][i1], &o = S[L][io];
          int p2 = (l2 & 1) ? -1 : 1;
          if (std::abs(a.l - l2) <= o.l && o.l <= a.l + l2 && o.p == a.p * p2) paths[L - 1].push_back({i1, l2, io});
        }
}

int al_build_tp_tables(allegro_model* m, const std::vector<std::vector<float>>& alphas) {
  std::vector<std::vector<Irrep>> S;
  std::vector<std::vector<TPLayerHost::Path>> paths;
  al_enumerate(m->lmax, m->NL, S, paths);
  m->tp_host.assign(m->NL, TPLayerHost());
  m->D.clear();
  for (auto& s : S) {
    int dsum = 0;
    for (auto& ir : s) dsum += 2 * ir.l + 1;
    m->D.push_back(dsum);
  }
  // V^0 layout maps
  m->v0_l.clear(); m->v0_y.clear();
  for (auto& ir : S[0])
    for (int k = 0; k < 2 * ir.l + 1; ++k) { m->v0_l.push_back(ir.l); m->v0_y.push_back(ir.l * ir.l + k); }
  for (int L = 1; L <= m->NL; ++L) {
    TPLayerHost& t = m->tp_host[L - 1];
    t.in = S[L - 1]; t.out = S[L];
    t.Din = m->D[L - 1]; t.Dout = m->D[L]; t.Denv = m->Denv;
    t.paths = paths[L - 1];
    std::map<int, int> cnt;
    for (auto& p : t.paths) cnt[p.io]++;
    t.fan.clear();
    for (auto& p : t.paths) t.fan.push_back(cnt[p.io]);
    std::vector<int> off1, offo;
    { int o = 0; for (auto& ir : t.in) { off1.push_back(o); o += 2 * ir.l + 1; } }
    { int o = 0; for (auto& ir : t.out) { offo.push_back(o); o += 2 * ir.l + 1; } }
    // dense accumulate (blocks of different paths never overlap, but accumulate anyway)
    std::vector<double> K((size_t)t.Din * t.Denv * t.Dout, 0.0);
    for (size_t pi = 0; pi < t.paths.size(); ++pi) {
      auto& p = t.paths[pi];
      int l1 = t.in[p.i1].l, l2 = p.l2, lo = t.out[p.io].l;
      std::vector<double> C = real_cg_block(l1, l2, lo);
      double alpha = alphas.empty() ? 1.0 : (double)alphas[L - 1][pi];
      for (int a = 0; a < 2 * l1 + 1; ++a)
        for (int b = 0; b < 2 * l2 + 1; ++b)
          for (int c = 0; c < 2 * lo + 1; ++c) {
            double v = C[(a * (2 * l2 + 1) + b) * (2 * lo + 1) + c];
            if (v != 0.0) K[((size_t)(off1[p.i1] + a) * t.Denv + (l2 * l2 + b)) * t.Dout + offo[p.io] + c] += alpha * v;
          }
    }
    // sparse structure is taken from the CG pattern with alpha = 1 so it does not depend on weights
    // (an alpha that happens to be 0 keeps explicit zeros): rebuild pattern
    std::vector<char> pat((size_t)t.Din * t.Denv * t.Dout, 0);
    for (auto& p : t.paths) {
      int l1 = t.in[p.i1].l, l2 = p.l2, lo = t.out[p.io].l;
      std::vector<double> C = real_cg_block(l1, l2, lo);
      for (int a = 0; a < 2 * l1 + 1; ++a)
        for (int b = 0; b < 2 * l2 + 1; ++b)
          for (int c = 0; c < 2 * lo + 1; ++c)
            if (C[(a * (2 * l2 + 1) + b) * (2 * lo + 1) + c] != 0.0)
              pat[((size_t)(off1[p.i1] + a) * t.Denv + (l2 * l2 + b)) * t.Dout + offo[p.io] + c] = 1;
    }
    t.pair_a.clear(); t.pair_c.clear(); t.pair_ptr.assign(1, 0); t.ent_b.clear(); t.ent_val.clear();
    t.nnz = 0;
    // pairs ordered by (c, a) so that pairs of one output component are contiguous
    for (int c = 0; c < t.Dout; ++c)
      for (int a = 0; a < t.Din; ++a) {
        bool any = false;
        for (int b = 0; b < t.Denv; ++b)
          if (pat[((size_t)a * t.Denv + b) * t.Dout + c]) {
            any = true;
            t.ent_b.push_back(b);
            t.ent_val.push_back((float)K[((size_t)a * t.Denv + b) * t.Dout + c]);
            t.nnz++;
          }
        if (any) { t.pair_a.push_back(a); t.pair_c.push_back(c); t.pair_ptr.push_back((int)t.ent_b.size()); }
      }
    t.npairs = (int)t.pair_a.size();
    t.ent_idx.assign(t.nnz, 0);
    for (int p = 0; p < t.npairs; ++p)
      for (int k = t.pair_ptr[p]; k < t.pair_ptr[p + 1]; ++k) t.ent_idx[k] = t.pair_a[p] * t.Dout + t.pair_c[p];
    // packed entry lists sorted by c (already the entry order) and by a
    t.ce_pack.assign(t.nnz, 0); t.ce_val = t.ent_val; t.cent_ptr.assign(t.Dout + 1, 0);
    for (int p = 0; p < t.npairs; ++p)
      for (int k = t.pair_ptr[p]; k < t.pair_ptr[p + 1]; ++k) {
        t.ce_pack[k] = t.pair_a[p] | (t.pair_c[p] << 8) | (t.ent_b[k] << 16);
        t.cent_ptr[t.pair_c[p] + 1]++;
      }
    for (int c = 0; c < t.Dout; ++c) t.cent_ptr[c + 1] += t.cent_ptr[c];
    t.aent_ptr.assign(t.Din + 1, 0);
    for (int k = 0; k < t.nnz; ++k) t.aent_ptr[(t.ce_pack[k] & 255) + 1]++;
    for (int a = 0; a < t.Din; ++a) t.aent_ptr[a + 1] += t.aent_ptr[a];
    t.ae_pack.assign(t.nnz, 0); t.ae_val.assign(t.nnz, 0.f);
    {
      std::vector<int> af(t.aent_ptr.begin(), t.aent_ptr.end() - 1);
      for (int k = 0; k < t.nnz; ++k) { int a = t.ce_pack[k] & 255; t.ae_pack[af[a]] = t.ce_pack[k]; t.ae_val[af[a]++] = t.ce_val[k]; }
    }
    // dense pair table (a-major, c-minor), empty pairs have zero length
    t.dp_ptr.assign((size_t)t.Din * t.Dout + 1, 0); t.dp_b.clear(); t.dp_val.clear();
    for (int a = 0; a < t.Din; ++a)
      for (int c = 0; c < t.Dout; ++c) {
        for (int b = 0; b < t.Denv; ++b)
          if (pat[((size_t)a * t.Denv + b) * t.Dout + c]) {
            t.dp_b.push_back(b);
            t.dp_val.push_back((float)K[((size_t)a * t.Denv + b) * t.Dout + c]);
          }
        t.dp_ptr[(size_t)a * t.Dout + c + 1] = (int)t.dp_b.size();
      }
    // CSR over c and over a
    t.c_ptr.assign(t.Dout + 1, 0); t.a_ptr.assign(t.Din + 1, 0); t.b_ptr.assign(t.Denv + 1, 0);
    for (int p = 0; p < t.npairs; ++p) { t.c_ptr[t.pair_c[p] + 1]++; t.a_ptr[t.pair_a[p] + 1]++; }
    for (int c = 0; c < t.Dout; ++c) t.c_ptr[c + 1] += t.c_ptr[c];
    for (int a = 0; a < t.Din; ++a) t.a_ptr[a + 1] += t.a_ptr[a];
    t.c_a.assign(t.npairs, 0); t.c_p.assign(t.npairs, 0); t.a_c.assign(t.npairs, 0); t.a_p.assign(t.npairs, 0);
    {
      std::vector<int> cf(t.c_ptr.begin(), t.c_ptr.end() - 1), af(t.a_ptr.begin(), t.a_ptr.end() - 1);
      for (int p = 0; p < t.npairs; ++p) {
        int c = t.pair_c[p], a = t.pair_a[p];
        t.c_a[cf[c]] = a; t.c_p[cf[c]++] = p;
        t.a_c[af[a]] = c; t.a_p[af[a]++] = p;
      }
    }
    for (int p = 0; p < t.npairs; ++p)
      for (int k = t.pair_ptr[p]; k < t.pair_ptr[p + 1]; ++k) t.b_ptr[t.ent_b[k] + 1]++;
    for (int b = 0; b < t.Denv; ++b) t.b_ptr[b + 1] += t.b_ptr[b];
    t.b_p.assign(t.nnz, 0); t.b_val.assign(t.nnz, 0.f);
    {
      std::vector<int> bf(t.b_ptr.begin(), t.b_ptr.end() - 1);
      for (int p = 0; p < t.npairs; ++p)
        for (int k = t.pair_ptr[p]; k < t.pair_ptr[p + 1]; ++k) {
          int b = t.ent_b[k];
          t.b_p[bf[b]] = p; t.b_val[bf[b]++] = t.ent_val[k];
        }
    }
  }
  return ALLEGRO_OK;
}
