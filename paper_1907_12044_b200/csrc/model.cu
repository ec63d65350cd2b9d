// model.cu -- host-side builder of the workload's Hamiltonian as an MPO: the
// Frenkel-Holstein model of PAPER.md:312-318, Eq. 45,
//     H = sum_m E_m a+_m a_m + sum_{m != n} J_mn a+_m a_n
//       + sum_{m,l} w_ml (b+_ml b_ml + 1/2) + sum_{m,l} g_ml w_ml (b+_ml + b_ml) a+_m a_m ,
// in the form of Eq. 11.  No GPU work: plain host code, so that a user of the library can
// build the paper's workload without anything outside it.
//
// Construction: H is written as a list of one-site terms (site, O) and two-site terms
// (site a, A) x (site b > a, B); two-site terms that share their left factor (a, A) share one bond channel
// from a to the right-most b.  The MPO is the finite-state machine over the channels
//   "done"  (a complete term sits to the left; identities follow),
//   "start" (only identities so far),
//   one channel per open group (a, A),
// with transitions start -> done (one-site terms), start -> group (A at site a), group -> done (B at site b),
// and identities on every channel that passes a site.  Site tensors are real and mostly zero
// (SURVEY.md 8(c) c3).  Readings c1 (layouts A / B), c4 (g = sqrt(Huang-Rhys factor), zero-point term kept).
#include <cmath>
#include <map>
#include <vector>

#include "handle.cuh"

namespace {

typedef std::vector<double> Mat;     // d x d, row-major [out][in]

Mat mat_zero(int d) { return Mat((size_t)d * d, 0.0); }
Mat mat_eye(int d) { Mat m = mat_zero(d); for (int i = 0; i < d; i++) m[(size_t)i * d + i] = 1.0; return m; }
void mat_axpy(Mat &y, double a, const Mat &x) { for (size_t i = 0; i < y.size(); i++) y[i] += a * x[i]; }

struct Group {                       // two-site terms sharing the left factor
  int site;                          // a
  Mat A;
  std::vector<std::pair<int, Mat>> closers;   // (b, coefficient * B)
  int last = -1;                     // right-most b
};

struct TermList {
  std::vector<int> dims;
  std::vector<Mat> onsite;           // sum of the one-site terms of every site
  std::vector<Group> groups;
};

// phonon operators in the number basis truncated to n_ph states
Mat number_plus_half(int n) { Mat m = mat_zero(n); for (int v = 0; v < n; v++) m[(size_t)v * n + v] = v + 0.5; return m; }
Mat displacement(int n) {            // b+ + b
  Mat m = mat_zero(n);
  for (int v = 1; v < n; v++) { m[(size_t)(v - 1) * n + v] = std::sqrt((double)v); m[(size_t)v * n + (v - 1)] = std::sqrt((double)v); }
  return m;
}

TermList vibronic_terms(int layout, int n_el, int n_modes, int n_ph, const double *E, const double *J, const double *omega,
                        const double *S, double unit) {
  TermList t;
  if (layout == 0) {
    // layout A: one electronic site of dimension n_el (single-exciton sector), then the modes, state-major
    t.dims.push_back(n_el);
    for (int k = 0; k < n_el * n_modes; k++) t.dims.push_back(n_ph);
    for (size_t i = 0; i < t.dims.size(); i++) t.onsite.push_back(mat_zero(t.dims[i]));
    for (int m = 0; m < n_el; m++)
      for (int q = 0; q < n_el; q++) t.onsite[0][(size_t)m * n_el + q] = unit * (m == q ? E[m] : J[m * n_el + q]);
    for (int m = 0; m < n_el; m++) {
      Group g; g.site = 0; g.A = mat_zero(n_el); g.A[(size_t)m * n_el + m] = 1.0;       // |m><m|
      for (int l = 0; l < n_modes; l++) {
        const int s = 1 + m * n_modes + l;
        const double w = unit * omega[m * n_modes + l], gc = std::sqrt(S[m * n_modes + l]);
        mat_axpy(t.onsite[s], w, number_plus_half(n_ph));
        Mat B = mat_zero(n_ph); mat_axpy(B, gc * w, displacement(n_ph));
        g.closers.push_back({s, B});
        g.last = s;
      }
      if (!g.closers.empty()) t.groups.push_back(g);
    }
  } else {
    // layout B (the paper's): a two-level site per electronic state, followed by its modes
    std::vector<int> el(n_el);
    for (int m = 0; m < n_el; m++) { el[m] = (int)t.dims.size(); t.dims.push_back(2); for (int l = 0; l < n_modes; l++) t.dims.push_back(n_ph); }
    for (size_t i = 0; i < t.dims.size(); i++) t.onsite.push_back(mat_zero(t.dims[i]));
    Mat up = mat_zero(2), dn = mat_zero(2), nn = mat_zero(2);
    up[2] = 1.0;                    // a+ : |0> -> |1>   ([out][in] = [1][0])
    dn[1] = 1.0;                    // a
    nn[3] = 1.0;                    // a+ a
    for (int m = 0; m < n_el; m++) {
      mat_axpy(t.onsite[el[m]], unit * E[m], nn);
      Group gp, gm, gn;
      gp.site = gm.site = gn.site = el[m];
      gp.A = up; gm.A = dn; gn.A = nn;
      for (int q = m + 1; q < n_el; q++) {
        const double j = unit * J[m * n_el + q];
        if (j == 0.0) continue;
        Mat Bd = mat_zero(2), Bu = mat_zero(2);
        mat_axpy(Bd, j, dn); mat_axpy(Bu, j, up);
        gp.closers.push_back({el[q], Bd}); gp.last = el[q];      // J a+_m a_q
        gm.closers.push_back({el[q], Bu}); gm.last = el[q];      // J a_m a+_q
      }
      for (int l = 0; l < n_modes; l++) {
        const int s = el[m] + 1 + l;
        const double w = unit * omega[m * n_modes + l], gc = std::sqrt(S[m * n_modes + l]);
        mat_axpy(t.onsite[s], w, number_plus_half(n_ph));
        Mat B = mat_zero(n_ph); mat_axpy(B, gc * w, displacement(n_ph));
        gn.closers.push_back({s, B}); gn.last = s;
      }
      if (!gp.closers.empty()) t.groups.push_back(gp);
      if (!gm.closers.empty()) t.groups.push_back(gm);
      if (!gn.closers.empty()) t.groups.push_back(gn);
    }
  }
  return t;
}

}  // namespace

extern "C" {

int tdvp_build_vibronic_mpo(int layout, int n_el, int n_modes, int n_ph, const double *E, const double *J, const double *omega,
                            const double *huang_rhys, double energy_unit, int *n_sites, int *phys_dim, int *mpo_bond,
                            tdvp_c128 *const *mpo) {
  if ((layout != 0 && layout != 1) || n_el < 1 || n_modes < 0 || n_ph < 1 || !E || !J || (n_modes > 0 && (!omega || !huang_rhys)) || !n_sites)
    return set_err(nullptr, TDVP_EINVAL, "tdvp_build_vibronic_mpo: bad argument");
  for (int k = 0; k < n_el * n_modes; k++)
    if (!(huang_rhys[k] >= 0.0)) return set_err(nullptr, TDVP_EINVAL, "tdvp_build_vibronic_mpo: Huang-Rhys factors must be >= 0");
  const TermList t = vibronic_terms(layout, n_el, n_modes, n_ph, E, J, omega, huang_rhys, energy_unit);
  const int n = (int)t.dims.size();
  *n_sites = n;
  // channels on bond b (between sites b - 1 and b): b = 0: [start]; b = n: [done]; else [done, start, open groups]
  std::vector<std::vector<int>> open(n + 1);        // group indices alive on bond b: site < b <= last
  for (int b = 1; b < n; b++)
    for (size_t g = 0; g < t.groups.size(); g++)
      if (t.groups[g].site < b && b <= t.groups[g].last) open[b].push_back((int)g);
  auto bond_dim = [&](int b) { return (b == 0 || b == n) ? 1 : 2 + (int)open[b].size(); };
  if (phys_dim) for (int i = 0; i < n; i++) phys_dim[i] = t.dims[i];
  if (mpo_bond) for (int b = 0; b <= n; b++) mpo_bond[b] = bond_dim(b);
  if (!mpo) return TDVP_OK;                         // size query
  for (int i = 0; i < n; i++) {
    if (!mpo[i]) return set_err(nullptr, TDVP_EINVAL, "tdvp_build_vibronic_mpo: null site tensor");
    const int d = t.dims[i], Dl = bond_dim(i), Dr = bond_dim(i + 1);
    tdvp_c128 *W = mpo[i];
    for (size_t e = 0; e < (size_t)Dl * d * d * Dr; e++) { W[e].re = 0.0; W[e].im = 0.0; }
    // channel indices: left bond i, right bond i + 1
    const int l_done = (i == 0) ? -1 : 0, l_start = (i == 0) ? 0 : 1;
    const int r_done = (i == n - 1) ? 0 : 0, r_start = (i == n - 1) ? -1 : 1;
    auto l_group = [&](int g) { for (size_t k = 0; k < open[i].size(); k++) if (open[i][k] == g) return 2 + (int)k; return -1; };
    auto r_group = [&](int g) { if (i == n - 1) return -1; for (size_t k = 0; k < open[i + 1].size(); k++) if (open[i + 1][k] == g) return 2 + (int)k; return -1; };
    auto add = [&](int wl, int wr, const Mat &O, double c) {
      if (wl < 0 || wr < 0) return;
      for (int p = 0; p < d; p++)
        for (int s = 0; s < d; s++) W[(((size_t)wl * d + p) * d + s) * Dr + wr].re += c * O[(size_t)p * d + s];
    };
    const Mat I = mat_eye(d);
    add(l_done, r_done, I, 1.0);                    // done -> done
    add(l_start, r_start, I, 1.0);                  // start -> start
    add(l_start, r_done, t.onsite[i], 1.0);         // one-site terms
    for (size_t g = 0; g < t.groups.size(); g++) {
      const Group &G = t.groups[g];
      if (G.site == i) add(l_start, r_group((int)g), G.A, 1.0);                  // open
      if (G.site < i && i <= G.last) {
        for (const auto &c : G.closers) if (c.first == i) add(l_group((int)g), r_done, c.second, 1.0);   // close
        if (i < G.last) add(l_group((int)g), r_group((int)g), I, 1.0);           // pass
      }
    }
  }
  return TDVP_OK;
}

}  // extern "C"
