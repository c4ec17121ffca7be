/*
 * ckb_pack.cu -- host-side validation and packing of a mechanism into the device tables of
 * ckb_tables.h.  No kernels here.
 */
#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <map>
#include <numeric>
#include <utility>
#include <vector>

#include "ckb_host.h"

namespace ckb_host {

namespace {

constexpr double RC_CAL = 1.98720425864; /* R20: cal/(mol K) */

inline unsigned long long dbits(double x) {
  unsigned long long u;
  std::memcpy(&u, &x, 8);
  return u;
}

}  // namespace

int parse_mechanism(const ckb_mech_desc *d, Parsed &P, const FoDesc *fo) {
  const int K = d->n_species, R = d->n_reactions, R3 = d->n_third_body;
  if (K < 1 || R < 0 || R3 < 0) return CKB_EINVAL;
  if (!d->mol_weight || !d->nasa) return CKB_EINVAL;
  if (R > 0 && (!d->arr_A || !d->arr_beta || !d->arr_E || !d->reac_ptr || !d->prod_ptr)) return CKB_EINVAL;
  if (R3 > 0 && (!d->tb_reaction || !d->tb_ptr)) return CKB_EINVAL;
  if (K > 254) return CKB_EUNSUPPORTED;
  for (int k = 0; k < K; k++) {
    if (!(d->mol_weight[k] > 0.0) || !std::isfinite(d->mol_weight[k])) return CKB_EINVAL;
    for (int q = 0; q < 6; q++)
      if (!std::isfinite(d->nasa[7 * (size_t)k + q])) return CKB_EINVAL;
  }
  if (R > 0 && (d->reac_ptr[0] != 0 || d->prod_ptr[0] != 0)) return CKB_EINVAL;
  if (R3 > 0 && d->tb_ptr[0] != 0) return CKB_EINVAL;
  P.K = K;
  P.R = R;
  P.W.assign(d->mol_weight, d->mol_weight + K);
  P.nasa.assign(d->nasa, d->nasa + 7 * (size_t)K);
  if (R > 0) {
    P.A.assign(d->arr_A, d->arr_A + R);
    P.beta.assign(d->arr_beta, d->arr_beta + R);
    P.E.assign(d->arr_E, d->arr_E + R);
  }
  std::vector<Rx> &rx = P.rx;
  rx.resize(R);
  for (int j = 0; j < R; j++) {
    if (d->reac_ptr[j + 1] < d->reac_ptr[j] || d->prod_ptr[j + 1] < d->prod_ptr[j]) return CKB_EINVAL;
    if (!(d->arr_A[j] >= 0.0) || !std::isfinite(d->arr_A[j]) || !std::isfinite(d->arr_beta[j]) ||
        !std::isfinite(d->arr_E[j]))
      return CKB_EINVAL;
    for (int side = 0; side < 2; side++) {
      const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
      const int32_t *sp = side ? d->prod_species : d->reac_species;
      const int32_t *nu = side ? d->prod_nu : d->reac_nu;
      std::vector<int> &mol = side ? rx[j].prod : rx[j].reac;
      if (ptr[j + 1] > ptr[j] && (!sp || !nu)) return CKB_EINVAL;
      for (int e = ptr[j]; e < ptr[j + 1]; e++) {
        if (sp[e] < 0 || sp[e] >= K || nu[e] < 1) return CKB_EINVAL;
        if (nu[e] > 3) return CKB_EUNSUPPORTED;
        for (int q = 0; q < nu[e]; q++) mol.push_back(sp[e]);
      }
      if (mol.size() > 3) return CKB_EUNSUPPORTED;
      std::sort(mol.begin(), mol.end());
    }
  }
  /* third-body efficiency sets, deduplicated */
  std::map<std::vector<std::pair<int, double>>, int> set_id;
  for (int r = 0; r < R3; r++) {
    const int j = d->tb_reaction[r];
    if (j < 0 || j >= R || rx[j].tbset >= 0) return CKB_EINVAL;
    if (d->tb_ptr[r + 1] < d->tb_ptr[r]) return CKB_EINVAL;
    std::map<int, double> eff; /* a species listed twice: the last entry wins */
    for (int e = d->tb_ptr[r]; e < d->tb_ptr[r + 1]; e++) {
      if (!d->tb_species || !d->tb_eff) return CKB_EINVAL;
      if (d->tb_species[e] < 0 || d->tb_species[e] >= K || !std::isfinite(d->tb_eff[e])) return CKB_EINVAL;
      eff[d->tb_species[e]] = d->tb_eff[e];
    }
    std::vector<std::pair<int, double>> key(eff.begin(), eff.end());
    auto it = set_id.find(key);
    if (it == set_id.end()) {
      it = set_id.emplace(key, (int)P.sets.size()).first;
      P.sets.push_back(key);
    }
    rx[j].tbset = it->second;
  }
  /* R31: a fall-off reaction owns an efficiency set (its third-body efficiencies if it has them, else all 1), whose
   * "[M]" the kernels replace by the blending factor P_r/(1+P_r) F -- a per-reaction multiplier like [M] itself */
  if (fo && fo->n > 0) {
    if (!fo->reaction || !fo->low3 || !fo->troe4) return CKB_EINVAL;
    std::vector<char> seen(R, 0);
    for (int i = 0; i < fo->n; i++) {
      const int j = fo->reaction[i];
      if (j < 0 || j >= R || seen[j]) return CKB_EINVAL;
      seen[j] = 1;
      const double A0 = fo->low3[3 * i], b0 = fo->low3[3 * i + 1], E0 = fo->low3[3 * i + 2];
      const double *tr = fo->troe4 + 4 * (size_t)i;
      if (!(A0 > 0.0) || !std::isfinite(A0) || !std::isfinite(b0) || !std::isfinite(E0) || !(d->arr_A[j] > 0.0))
        return CKB_EINVAL;
      Parsed::Fo f;
      f.dlnA = std::log(A0) - std::log(d->arr_A[j]);
      f.dbeta = b0 - d->arr_beta[j];
      f.dtheta = (E0 - d->arr_E[j]) / RC_CAL;
      if (tr[0] != tr[0]) {
        f.kind = 1;
      } else {
        if (!std::isfinite(tr[0]) || !(tr[1] > 0.0) || !(tr[2] > 0.0) || tr[3] != tr[3]) return CKB_EINVAL;
        f.kind = std::isfinite(tr[3]) ? 2 : 3;
        f.a = tr[0];
        f.invT3 = 1.0 / tr[1]; /* 1/inf = 0: exp(-T/inf) = 1 */
        f.invT1 = 1.0 / tr[2];
        f.T2 = std::isfinite(tr[3]) ? tr[3] : 0.0;
      }
      std::vector<std::pair<int, double>> key;
      if (rx[j].tbset >= 0) key = P.sets[rx[j].tbset];
      rx[j].tbset = (int)P.sets.size();
      P.sets.push_back(key);
      P.fo.resize(P.sets.size());
      P.fo.back() = f;
    }
  }
  if (P.sets.size() > 65000) return CKB_EUNSUPPORTED;
  if (!P.fo.empty()) {
    /* Efficiency sets in the order Troe, Lindemann, ordinary: the lane-distributed kernels evaluate the blending factors
     * set round by set round, each lane its own set -- grouped like this the fall-off sets fill whole rounds with lanes
     * that all do the same work, and the rounds of ordinary sets skip the pass (53/634 with 51 fall-off reactions: 2 busy
     * rounds instead of 4 half-idle ones). */
    P.fo.resize(P.sets.size());
    std::vector<int> order(P.sets.size()), new_id(P.sets.size());
    std::iota(order.begin(), order.end(), 0);
    auto rank = [&](int t) { return P.fo[t].kind >= 2 ? 0 : P.fo[t].kind == 1 ? 1 : 2; };
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return rank(a) < rank(b); });
    std::vector<std::vector<std::pair<int, double>>> sets2(P.sets.size());
    std::vector<Parsed::Fo> fo2(P.sets.size());
    for (size_t q = 0; q < order.size(); q++) {
      new_id[order[q]] = (int)q;
      sets2[q] = P.sets[order[q]];
      fo2[q] = P.fo[order[q]];
    }
    P.sets.swap(sets2);
    P.fo.swap(fo2);
    for (int j = 0; j < R; j++)
      if (rx[j].tbset >= 0) rx[j].tbset = new_id[rx[j].tbset];
  }

  /* fuse forward / reverse reactions over the same species (and the same third body) into one slot */
  typedef std::pair<std::pair<std::vector<int>, std::vector<int>>, int> Key;
  std::map<Key, std::vector<int>> waiting; /* key of an unpaired reaction -> its slot index */
  for (int j = 0; j < R; j++) {
    Key rev{{rx[j].prod, rx[j].reac}, rx[j].tbset};
    auto it = waiting.find(rev);
    if (it != waiting.end() && !it->second.empty()) {
      P.slots[it->second.back()].r = j;
      it->second.pop_back();
    } else {
      Key self{{rx[j].reac, rx[j].prod}, rx[j].tbset};
      waiting[self].push_back((int)P.slots.size());
      P.slots.push_back({j, -1});
    }
  }
  /* species-major gather rows: net coefficient of the slot's forward direction (Eq. 3) */
  P.rows.assign(K, {});
  for (int s = 0; s < (int)P.slots.size(); s++) {
    const Rx &f = rx[P.slots[s].f];
    std::map<int, int> net;
    for (int k : f.prod) net[k] += 1;
    for (int k : f.reac) net[k] -= 1;
    for (auto &kv : net)
      if (kv.second != 0) P.rows[kv.first].push_back({s, kv.second});
  }
  /* algorithmic flops per f(y), DESIGN.md 7.2 (FMA = 2, exp = 30, log = 46, division = 36) */
  double F = 0.0;
  for (int j = 0; j < R; j++) {
    F += 4.0 + 30.0;                                                 /* Eq. 5 */
    F += (double)rx[j].reac.size() + (rx[j].tbset >= 0 ? 1.0 : 0.0); /* Eq. 4 */
    for (int side = 0; side < 2; side++) {                           /* Eq. 3 */
      const int32_t *ptr = side ? d->prod_ptr : d->reac_ptr;
      const int32_t *nu = side ? d->prod_nu : d->reac_nu;
      for (int e = ptr[j]; e < ptr[j + 1]; e++) F += nu[e] == 1 ? 1.0 : 2.0;
    }
  }
  for (int r = 0; r < R3; r++) F += 2.0 * (d->tb_ptr[r + 1] - d->tb_ptr[r]) + 1.0;
  F += 27.0 * K + 46.0 + 3.0 * 36.0; /* thermo, Eq. 2, Eq. 6, rho, ln T, 1/T */
  for (auto &f : P.fo) {             /* R31: k_0 (one exp), P_r, P_r/(1+P_r); Troe: F_cent, two log10, 10^x */
    if (f.kind >= 1) F += 4.0 + 30.0 + 2.0 + 36.0;
    if (f.kind >= 2) F += (f.kind == 2 ? 3.0 : 2.0) * 32.0 + 2.0 * 46.0 + 12.0 + 36.0 + 36.0 + 30.0;
  }
  P.flops_per_rhs = F;
  return CKB_OK;
}

/* RKC coefficients of an s-stage step, Eq. 22-26 with R8 (w0 = 1 + (2/13)/s^2), R9
 * (a_j = 1 - b_j T_j(w0)) and R10 (b_0 = b_1 = b_2).  out: mu~_1, then (mu_j, nu_j, mu~_j, gamma~_j), j = 2..s. */
void rkc_stage_coefficients(int s, double *mut1, double *stages) {
  std::vector<double> T(s + 1), dT(s + 1), d2T(s + 1), b(s + 1), a(s + 1);
  const double w0 = 1.0 + (2.0 / 13.0) / ((double)s * (double)s);
  T[0] = 1.0; T[1] = w0; dT[0] = 0.0; dT[1] = 1.0; d2T[0] = 0.0; d2T[1] = 0.0;
  for (int j = 2; j <= s; j++) {
    T[j] = 2.0 * w0 * T[j - 1] - T[j - 2];
    dT[j] = 2.0 * T[j - 1] + 2.0 * w0 * dT[j - 1] - dT[j - 2];
    d2T[j] = 4.0 * dT[j - 1] + 2.0 * w0 * d2T[j - 1] - d2T[j - 2];
  }
  const double w1 = dT[s] / d2T[s];
  for (int j = 2; j <= s; j++) b[j] = d2T[j] / (dT[j] * dT[j]);
  b[0] = b[2];
  b[1] = b[2];
  for (int j = 0; j <= s; j++) a[j] = 1.0 - b[j] * T[j];
  *mut1 = b[1] * w1;
  for (int j = 2; j <= s; j++) {
    const double mut = 2.0 * b[j] * w1 / b[j - 1];
    stages[4 * (j - 2) + 0] = 2.0 * b[j] * w0 / b[j - 1];
    stages[4 * (j - 2) + 1] = -b[j] / b[j - 2];
    stages[4 * (j - 2) + 2] = mut;
    stages[4 * (j - 2) + 3] = -a[j - 1] * mut;
  }
}

/* ------------------------------------------------------------------------------------------------
 * Bank-conflict-aware scheduling.  Shared memory has 32 four-byte banks; a 64-bit warp
 * access is served half-warp by half-warp, and is conflict free when the 16 lanes of a half-warp touch 16
 * distinct bank pairs (or the same address).  Where a lane reads is table data, so the packer chooses it:
 *   - place_slots(): which reaction slot each lane evaluates in each round, and in which order it reads the
 *     molecules of a side, so that the concentration reads of a half-warp collide as little as possible;
 *   - colour_gather(): the order in which each lane walks its gather row, by edge-colouring the bipartite
 *     multigraph (lane, bank pair of q_s): every step reads 16 distinct bank pairs per half-warp (Koenig:
 *     max-degree many steps suffice).
 * Both only reorder commutative products / sums: the result changes by rounding only.
 * ---------------------------------------------------------------------------------------------- */
namespace {

struct Placed {
  int slot = -1;          /* index into Parsed::slots, -1 = padding */
  int a[3] = {0, 0, 0};   /* components read as reactant molecules (0 = none -> C_0 = 1) */
  int b[3] = {0, 0, 0};   /* components read as product molecules */
};

/* greedy: fill rounds position by position with the remaining slot (and molecule order) that adds the fewest
 * bank-pair collisions to its half-warp's six concentration reads */
std::vector<Placed> place_slots(const Parsed &P, const std::vector<int> &comp_of_sp, int L, int NSR, bool optimise) {
  const int NS = (int)P.slots.size();
  std::vector<Placed> out((size_t)NSR * L);
  auto comps = [&](int s, int a[3], int b[3]) {
    const Rx &x = P.rx[P.slots[s].f];
    const bool rev = P.slots[s].r >= 0;
    for (int q = 0; q < 3; q++) {
      a[q] = q < (int)x.reac.size() ? comp_of_sp[x.reac[q]] : 0;
      /* a slot without reverse multiplies k_r = 0 by 1, never by a concentration */
      b[q] = (rev && q < (int)x.prod.size()) ? comp_of_sp[x.prod[q]] : 0;
    }
  };
  if (!optimise || L < 16) {
    std::vector<int> order(NS);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int u, int v) {
      auto c = [&](int s) {
        const Rx &x = P.rx[P.slots[s].f];
        return (x.reac.size() > 2 || (P.slots[s].r >= 0 && x.prod.size() > 2)) ? 0 : (x.tbset >= 0 ? 1 : 2);
      };
      return c(u) < c(v);
    });
    for (int q = 0; q < NS; q++) {
      out[q].slot = order[q];
      comps(order[q], out[q].a, out[q].b);
      std::sort(out[q].a, out[q].a + 3, std::greater<int>()); /* present molecules first */
      std::sort(out[q].b, out[q].b + 3, std::greater<int>());
    }
    return out;
  }
  std::vector<char> used(NS, 0);
  std::vector<int> cls(NS, 2);
  for (int s = 0; s < NS; s++) {
    const Rx &x = P.rx[P.slots[s].f];
    if (x.reac.size() > 2 || (P.slots[s].r >= 0 && x.prod.size() > 2)) cls[s] = 0;
    else if (x.tbset >= 0) cls[s] = 1;
  }
  int left = NS;
  for (int r = 0; r < NSR && left > 0; r++) {
    for (int h = 0; h < L / 16 && left > 0; h++) {
      /* comp_at[k][bp] = component already read through bank pair bp by instruction k in this half-warp (0 = free) */
      int comp_at[6][16];
      for (auto &row : comp_at)
        for (int &v : row) v = 0;
      for (int l = 0; l < 16 && left > 0; l++) {
        int best = -1, best_cost = 1 << 30, best_a[3] = {0, 0, 0}, best_b[3] = {0, 0, 0};
        /* slots are handed out class by class (third molecule first, then third body, then the rest), so that
           whole rounds can skip the reads they do not need (per-round flags) */
        int cur_class = 3;
        for (int s = 0; s < NS; s++)
          if (!used[s]) cur_class = std::min(cur_class, cls[s]);
        for (int s = 0; s < NS && best_cost > 0; s++) {
          if (used[s] || cls[s] != cur_class) continue;
          int a[3], b[3];
          comps(s, a, b);
          std::sort(a, a + 3, std::greater<int>());
          std::sort(b, b + 3, std::greater<int>());
          /* try every order of the molecules on each side */
          const int na = (a[0] != 0) + (a[1] != 0) + (a[2] != 0), nb = (b[0] != 0) + (b[1] != 0) + (b[2] != 0);
          int pa[3] = {a[0], a[1], a[2]};
          do {
            int ca = 0;
            for (int q = 0; q < 3; q++)
              if (pa[q] && comp_at[q][pa[q] & 15] && comp_at[q][pa[q] & 15] != pa[q]) ca++;
            int pb[3] = {b[0], b[1], b[2]};
            do {
              int cb = 0;
              for (int q = 0; q < 3; q++)
                if (pb[q] && comp_at[3 + q][pb[q] & 15] && comp_at[3 + q][pb[q] & 15] != pb[q]) cb++;
              if (ca + cb < best_cost) {
                best_cost = ca + cb;
                best = s;
                for (int q = 0; q < 3; q++) { best_a[q] = pa[q]; best_b[q] = pb[q]; }
              }
            } while (std::prev_permutation(pb, pb + nb));
          } while (std::prev_permutation(pa, pa + na));
        }
        Placed &pl = out[(size_t)r * L + h * 16 + l];
        pl.slot = best;
        for (int q = 0; q < 3; q++) {
          pl.a[q] = best_a[q];
          pl.b[q] = best_b[q];
          if (best_a[q] && !comp_at[q][best_a[q] & 15]) comp_at[q][best_a[q] & 15] = best_a[q];
          if (best_b[q] && !comp_at[3 + q][best_b[q] & 15]) comp_at[3 + q][best_b[q] & 15] = best_b[q];
        }
        used[best] = 1;
        left--;
      }
    }
  }
  return out;
}

struct GEntry { int pos, coef; };

/* One gather level: rows[g] = entries lane g must sum.  Returns steps[t][g] (pos = -1: idle).  With
 * `optimise`, a proper edge colouring of (lane, pos mod 16) per half-warp; else row order. */
std::vector<std::vector<GEntry>> colour_gather(const std::vector<std::vector<GEntry>> &rows, int L, bool optimise,
                                               bool relaxed = false) {
  size_t maxlen = 0;
  for (auto &r : rows) maxlen = std::max(maxlen, r.size());
  if (!optimise || L < 16) {
    std::vector<std::vector<GEntry>> steps(maxlen, std::vector<GEntry>(L, GEntry{-1, 0}));
    for (int g = 0; g < L; g++)
      for (size_t t = 0; t < rows[g].size(); t++) steps[t][g] = rows[g][t];
    return steps;
  }
  if (relaxed) {
    /* As many steps as the longest row, not as the busiest bank pair: per step each lane takes, of the entries it has
     * left, the one whose bank pair is least used in this step by its half-warp, or waits if it can afford to.  A few
     * two-way conflicts remain (reported): a replay costs one cycle of the shared-memory pipe, a step an issue slot
     * per entry. */
    std::vector<std::vector<GEntry>> steps(maxlen, std::vector<GEntry>(L, GEntry{-1, 0}));
    for (int h = 0; h < L / 16; h++) {
      std::vector<std::vector<GEntry>> left(16);
      for (int l = 0; l < 16; l++) left[l] = rows[h * 16 + l];
      for (size_t t = 0; t < maxlen; t++) {
        int cnt[16] = {0};
        std::vector<int> order(16);
        std::iota(order.begin(), order.end(), 0);
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return left[a].size() > left[b].size(); });
        for (int l : order) {
          if (left[l].empty()) continue;
          const long slack = (long)(maxlen - t) - (long)left[l].size();
          size_t best = 0;
          for (size_t e = 1; e < left[l].size(); e++)
            if (cnt[left[l][e].pos & 15] < cnt[left[l][best].pos & 15]) best = e;
          if (cnt[left[l][best].pos & 15] > 0 && slack > 0) continue; /* wait for a free bank pair */
          cnt[left[l][best].pos & 15]++;
          steps[t][h * 16 + l] = left[l][best];
          left[l].erase(left[l].begin() + best);
        }
      }
    }
    return steps;
  }
  std::vector<std::vector<GEntry>> steps;
  for (int h = 0; h < L / 16; h++) {
    /* degrees */
    int deg_l[16] = {0}, deg_r[16] = {0};
    for (int l = 0; l < 16; l++)
      for (auto &e : rows[h * 16 + l]) { deg_l[l]++; deg_r[e.pos & 15]++; }
    int D = 0;
    for (int q = 0; q < 16; q++) D = std::max(D, std::max(deg_l[q], deg_r[q]));
    /* colour[c][l] = index into rows[h*16+l] of the edge of colour c at lane l, rcol[c][bp] = lane using bank pair bp */
    std::vector<std::vector<int>> at_l(D, std::vector<int>(16, -1)), at_r(D, std::vector<int>(16, -1));
    for (int l = 0; l < 16; l++) {
      const auto &row = rows[h * 16 + l];
      for (int ei = 0; ei < (int)row.size(); ei++) {
        const int bp = row[ei].pos & 15;
        int ca = 0, cb = 0;
        while (at_l[ca][l] >= 0) ca++;       /* colour free at the lane */
        while (at_r[cb][bp] >= 0) cb++;      /* colour free at the bank pair */
        if (ca != cb) {
          /* flip the ca/cb alternating path that starts at bank pair bp (it has an edge of colour ca, none of cb) */
          int cur_bp = bp, c_have = ca, c_want = cb;
          std::vector<std::pair<int, int>> path; /* (lane, edge index) along the path */
          while (true) {
            const int ln = at_r[c_have][cur_bp];
            if (ln < 0) break;
            const int e2 = at_l[c_have][ln];
            path.push_back({ln, e2});
            /* next: at lane ln, the edge of colour c_want */
            const int e3 = at_l[c_want][ln];
            if (e3 < 0) break;
            path.push_back({ln, e3});
            cur_bp = rows[h * 16 + ln][e3].pos & 15;
          }
          /* remove the path's edges from the tables, then re-insert with swapped colours */
          std::vector<int> cols(path.size());
          for (size_t q = 0; q < path.size(); q++) cols[q] = (q % 2 == 0) ? c_have : c_want;
          for (size_t q = 0; q < path.size(); q++) {
            const int ln = path[q].first, e = path[q].second, b2 = rows[h * 16 + ln][e].pos & 15;
            at_l[cols[q]][ln] = -1;
            at_r[cols[q]][b2] = -1;
          }
          for (size_t q = 0; q < path.size(); q++) {
            const int ln = path[q].first, e = path[q].second, b2 = rows[h * 16 + ln][e].pos & 15;
            const int nc = (cols[q] == c_have) ? c_want : c_have;
            at_l[nc][ln] = e;
            at_r[nc][b2] = ln;
          }
          /* now ca is free at bp as well */
        }
        at_l[ca][l] = ei;
        at_r[ca][bp] = l;
      }
    }
    if ((int)steps.size() < D) steps.resize(D, std::vector<GEntry>(L, GEntry{-1, 0}));
    for (int c = 0; c < D; c++)
      for (int l = 0; l < 16; l++)
        if (at_l[c][l] >= 0) steps[c][h * 16 + l] = rows[h * 16 + l][at_l[c][l]];
  }
  return steps;
}

/* bank-pair collisions a schedule causes (excess wavefronts of 64-bit half-warp accesses), for the packing report */
int excess_wavefronts(const std::vector<int> &addr_of_lane /* L entries (L = 16 or 32), -1 = none */) {
  int excess = 0;
  for (int h = 0; h < (int)addr_of_lane.size() / 16; h++) {
    std::map<int, std::vector<int>> by_bp;
    for (int l = 0; l < 16; l++) {
      const int a = addr_of_lane[h * 16 + l];
      if (a < 0) continue;
      auto &v = by_bp[a & 15];
      if (std::find(v.begin(), v.end(), a) == v.end()) v.push_back(a);
    }
    int worst = 1;
    for (auto &kv : by_bp) worst = std::max(worst, (int)kv.second.size());
    excess += worst - 1;
  }
  return excess;
}

}  // namespace

/* entries of species k's Eq. 3 row as the lane-distributed gather counts them (|nu| > 1 entered |nu| times) */
static int row_entries(const Parsed &P, int k) {
  int len = 0;
  for (auto &sc : P.rows[k]) len += std::abs(sc.second);
  return len;
}

void component_order(const Parsed &P, std::vector<int> &sp_of_comp, std::vector<int> &comp_of_sp, int cap) {
  const int K = P.K, n = K + 1;
  sp_of_comp.assign(n, -1);
  comp_of_sp.assign(K, 0);
  std::vector<int> order(K);
  std::iota(order.begin(), order.end(), 0);
  if (cap > 0)
    std::stable_sort(order.begin(), order.end(),
                     [&](int a, int b) { return std::min(row_entries(P, a), cap) > std::min(row_entries(P, b), cap); });
  else
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return P.rows[a].size() > P.rows[b].size(); });
  for (int c = 1; c < n; c++) {
    sp_of_comp[c] = order[c - 1];
    comp_of_sp[order[c - 1]] = c;
  }
}

int pack_for(const Parsed &P, int L, Packed &out) {
  const int K = P.K, n = K + 1;
  const int G = (L == 1) ? 32 : 1; /* shared-memory interleave of the region (Sys::GI) */
  const int NS = (int)P.slots.size(), NTB = (int)P.sets.size();
  const int NV = pick_nv(L, n), NSR = (NS + L - 1) / L, NTBR = (NTB + L - 1) / L;
  if (NV < 0) return CKB_EUNSUPPORTED;
  int TBE = 0;
  for (auto &s : P.sets) TBE = std::max(TBE, (int)s.size());
  /* 16-bit region offsets, in bytes */
  if ((long long)(n + NTB + 1) * G * 8 > 65535 ||
      ((long long)NSR * L * (L == CKB_NEGQ_L ? 2 : 1) + (L > 1 ? CKB_ZERO_SLOTS : 0)) * G * 8 > 65535) /* q, -q and the 0.0 slots of idle entries */
    return CKB_EUNSUPPORTED;
  const bool optimise = true;

  /* Row splitting (lane-distributed mappings): the NV*L - n register slots of the last gather level that hold no
   * component take the TAILS of the longest Eq. 3 rows, so that no row is longer than cap = the (spare + 1)-th longest;
   * f(y) adds a tail to its component with one shuffle (DevMech::o_split). */
  const int spare = (L > 1) ? NV * L - n : 0;
  int cap = 0;
  if (spare > 0 && K > spare) {
    std::vector<int> lens(K);
    for (int k = 0; k < K; k++) lens[k] = row_entries(P, k);
    std::sort(lens.begin(), lens.end(), std::greater<int>());
    if (lens[0] > lens[spare] && lens[spare] >= 4) cap = lens[spare];
  }
  /* components: 0 = T, then species by decreasing (capped) gather-row length */
  std::vector<int> sp_of_comp, comp_of_sp;
  component_order(P, sp_of_comp, comp_of_sp, cap);
  std::vector<int> tail_slot(n, -1); /* component -> virtual slot (>= n) that holds the tail of its row */
  if (cap > 0) {
    int v = n;
    for (int c = 1; c < n && v < NV * L; c++)
      if (row_entries(P, sp_of_comp[c]) > cap) tail_slot[c] = v++;
  }
  /* which lane evaluates which slot, and the gather schedule of every level */
  const std::vector<Placed> placed = place_slots(P, comp_of_sp, L, NSR, optimise);
  std::vector<int> pos_of_slot(NS, -1);
  for (int q = 0; q < NSR * L; q++)
    if (placed[q].slot >= 0) pos_of_slot[placed[q].slot] = q;
  const int per_word_L = (L == 1) ? 1 : (L == CKB_NEGQ_L) ? 4 : 2; /* gather entries per 64-bit table word */
  std::vector<std::vector<std::vector<GEntry>>> sched(NV);
  std::vector<int> glen(NV, 0); /* 64-bit words per lane: two entries per word */
  for (int i = 0; i < NV; i++) {
    std::vector<std::vector<GEntry>> rows(L);
    for (int g = 0; g < L; g++) {
      const int c = g + L * i;
      if (c < 1) continue;
      int owner = c < n ? c : -1; /* a slot without a component holds the tail of some component's row */
      if (c >= n)
        for (int o = 1; o < n; o++)
          if (tail_slot[o] == c) owner = o;
      if (owner < 0) continue;
      std::vector<GEntry> all;
      for (auto &sc : P.rows[sp_of_comp[owner]]) {
        if (L == 1) {
          all.push_back(GEntry{pos_of_slot[sc.first], sc.second});
        } else { /* lane-distributed mappings apply the coefficient by where they read: |nu| > 1 is entered |nu| times */
          for (int rep = 0; rep < std::abs(sc.second); rep++)
            all.push_back(GEntry{pos_of_slot[sc.first], sc.second > 0 ? 1 : -1});
        }
      }
      if (c < n) { /* the head of the row (all of it unless it is split) */
        const size_t keep = (tail_slot[c] >= 0) ? (size_t)cap : all.size();
        rows[g].assign(all.begin(), all.begin() + std::min(keep, all.size()));
      } else {
        rows[g].assign(all.begin() + cap, all.end());
      }
    }
    sched[i] = colour_gather(rows, L, optimise, /*relaxed=*/true);
    glen[i] = (L == 1) ? (int)sched[i].size() : ((int)sched[i].size() + per_word_L - 1) / per_word_L;
  }
  const int gwords = std::accumulate(glen.begin(), glen.end(), 0);
  const int qcopies = (L == CKB_NEGQ_L) ? 2 : 1;
  const int s_tab = (L == 1) ? 12 : 48;

  ckb::DevMech &m = out.dm;
  m.K = K; m.n = n; m.L = L; m.NV = NV; m.NS = NS; m.NSR = NSR; m.NTB = NTB; m.NTBR = NTBR; m.TBE = TBE;
  int off = 0;
  auto take = [&off](size_t words) { /* every table starts on a 256-byte boundary: whole 128-byte lines per warp load */
    off = (off + 31) & ~31;
    int o = off;
    off += (int)words;
    return o;
  };
  m.o_sp = take((size_t)NV * CKB_SP_WORDS * L);
  m.o_sl = take((size_t)NSR * CKB_SL_WORDS * L);
  m.o_tb = take((size_t)NTBR * TBE * 2 * L);
  m.o_gat = take((size_t)gwords * L);
  m.o_glen = take(NV);
  m.o_rflag = off; off += NSR;
  m.o_perm = off; off += n;
  m.o_split = (cap > 0) ? take((size_t)NV * L) : 0;
  m.o_sp2 = P.nasa_hi.empty() ? 0 : take((size_t)NV * CKB_SP_WORDS * L);
  m.o_fo = P.fo.empty() ? 0 : take((size_t)NTBR * 8 * L);
  m.s_tab = s_tab;
  m.o_rkc = off; off += s_tab - 1;
  m.o_rkcs = off; off += 4 * (s_tab - 1) * s_tab / 2;
  m.words = off;
  std::vector<unsigned long long> &b = out.blob;
  b.assign((size_t)off, 0ull);
  auto putd = [&b](int o, double x) { b[(size_t)o] = dbits(x); };

  for (int c = 0; c < NV * L; c++) { /* species table; T and padding components keep zeros */
    const int i = c / L, g = c % L, base = m.o_sp + i * CKB_SP_WORDS * L + g;
    if (c >= 1 && c < n) {
      const int k = sp_of_comp[c];
      const double *a = &P.nasa[7 * (size_t)k];
      putd(base + CKB_SP_INVW * L, 1.0 / P.W[k]);
      putd(base + CKB_SP_W * L, P.W[k]);
      for (int q = 0; q < 5; q++) {
        putd(base + (CKB_SP_CP + q) * L, a[q]);
        putd(base + (CKB_SP_H + q) * L, a[q] / (double)(q + 1));
      }
      putd(base + (CKB_SP_H + 5) * L, a[5]);
    }
  }
  if (m.o_sp2) { /* R30: the high range, chosen on the device where T > T_mid (rows of T and padding: zeros) */
    for (int c = 1; c < n; c++) {
      const int i = c / L, g = c % L, base = m.o_sp2 + i * CKB_SP_WORDS * L + g;
      const int k = sp_of_comp[c];
      const double *a = &P.nasa_hi[7 * (size_t)k];
      putd(base + CKB_SP_INVW * L, P.Tmid[k]);
      for (int q = 0; q < 5; q++) {
        putd(base + (CKB_SP_CP + q) * L, a[q]);
        putd(base + (CKB_SP_H + q) * L, a[q] / (double)(q + 1));
      }
      putd(base + (CKB_SP_H + 5) * L, a[5]);
    }
  }
  for (int c = 0; c < n; c++) b[(size_t)m.o_perm + c] = (unsigned long long)(c == 0 ? 0 : 1 + sp_of_comp[c]);
  if (m.o_split)
    for (int c = 0; c < NV * L; c++) /* [level][lane] */
      b[(size_t)m.o_split + c] = (unsigned long long)(long long)((c < n && tail_slot[c] >= 0) ? tail_slot[c] % L : -1);

  const double LN_ZERO = -1.0e4; /* stands for ln 0: ckb_exp() returns ~1e-308 for it, no special case on the device */
  for (int q = 0; q < NSR * L; q++) {
    const int r = q / L, g = q % L, base = m.o_sl + r * CKB_SL_WORDS * L + g;
    const Placed &pl = placed[q];
    unsigned long long wa = 0, wb = 0;
    if (pl.slot >= 0) {
      const int f = P.slots[pl.slot].f, rv = P.slots[pl.slot].r;
      putd(base + CKB_SL_LNAF * L, P.A[f] > 0.0 ? std::log(P.A[f]) : LN_ZERO);
      putd(base + CKB_SL_BF * L, P.beta[f]);
      putd(base + CKB_SL_THF * L, P.E[f] / RC_CAL);
      putd(base + CKB_SL_LNAR * L, (rv >= 0 && P.A[rv] > 0.0) ? std::log(P.A[rv]) : LN_ZERO);
      putd(base + CKB_SL_BR * L, rv >= 0 ? P.beta[rv] : 0.0);
      putd(base + CKB_SL_THR * L, rv >= 0 ? P.E[rv] / RC_CAL : 0.0);
      for (int k = 0; k < 3; k++) {
        wa |= (unsigned long long)(pl.a[k] * G * 8) << (16 * k);
        wb |= (unsigned long long)(pl.b[k] * G * 8) << (16 * k);
      }
      const int ts = P.rx[f].tbset;
      wa |= (unsigned long long)((n + (ts >= 0 ? ts : NTB)) * G * 8) << 48;
    } else { /* padding slot: q = 0 */
      putd(base + CKB_SL_LNAF * L, LN_ZERO);
      putd(base + CKB_SL_LNAR * L, LN_ZERO);
      wa = (unsigned long long)((n + NTB) * G * 8) << 48;
    }
    b[(size_t)base + CKB_SL_IDXA * L] = wa;
    b[(size_t)base + CKB_SL_IDXB * L] = wb;
    /* round flags: 1 = some slot of the round reads a third molecule, 2 = some slot has a third body */
    if (pl.slot >= 0) {
      if (pl.a[2] || pl.b[2]) b[(size_t)m.o_rflag + r] |= 1ull;
      if (P.rx[P.slots[pl.slot].f].tbset >= 0) b[(size_t)m.o_rflag + r] |= 2ull;
    }
  }
  if (m.o_fo) { /* R31: per efficiency set, zeros (kind 0) for ordinary and padding sets */
    for (int t = 0; t < (int)P.fo.size(); t++) {
      const int r = t / L, g = t % L, base = m.o_fo + r * 8 * L + g;
      const Parsed::Fo &f = P.fo[t];
      const double w8[8] = {(double)f.kind, f.dlnA, f.dbeta, f.dtheta, f.a, f.invT3, f.invT1, f.T2};
      for (int x = 0; x < 8; x++) putd(base + x * L, w8[x]);
    }
  }
  for (int t = 0; t < NTBR * L; t++) { /* third-body sets, padded with (alpha - 1) = 0 on C_0 */
    const int r = t / L, g = t % L;
    for (int e = 0; e < TBE; e++) {
      const int base = m.o_tb + ((r * TBE + e) * 2) * L + g;
      if (t < NTB && e < (int)P.sets[t].size()) {
        putd(base, P.sets[t][e].second - 1.0);
        b[(size_t)base + L] = (unsigned long long)(comp_of_sp[P.sets[t][e].first] * G * 8);
      }
    }
  }
  { /* gather entries: L > 1: 16-bit byte offsets of q_s / -q_s, four per word; an idle lane reads the 0.0 slot of a bank
       pair nobody in its half-warp uses in that step.  L = 1: (double coefficient | q offset), one per word */
    int w0 = 0;
    out.gather_steps = 0;
    out.gather_excess_wavefronts = 0;
    for (int i = 0; i < NV; i++) {
      b[(size_t)m.o_glen + i] = (unsigned long long)glen[i];
      const int per_word = per_word_L;
      for (int t = 0; t < per_word * glen[i]; t++) {
        std::vector<int> addr(L >= 16 ? L : 0, -1);
        for (int g = 0; g < L; g++) {
          GEntry e = t < (int)sched[i].size() ? sched[i][t][g] : GEntry{-1, 0};
          if (e.pos < 0) {
            const bool zero_slot = L > 1; /* idle: + 0.0 from the zero slot of a bank pair nobody else reads */
            e.coef = zero_slot ? 1 : 0;
            e.pos = g % 16;
            if (L >= 16 && t < (int)sched[i].size()) {
              bool busy[16] = {false};
              for (int l = 0; l < 16; l++) {
                const GEntry &o = sched[i][t][(g / 16) * 16 + l];
                if (o.pos >= 0) busy[o.pos & 15] = true;
              }
              for (int l = 0; l < 16; l++)
                if (addr[(g / 16) * 16 + l] >= 0) busy[addr[(g / 16) * 16 + l] & 15] = true;
              for (int r0 = 0; r0 < 16; r0++)
                if (!busy[r0]) { e.pos = r0; break; }
            }
            if (zero_slot) e.pos = qcopies * NSR * L + ((e.pos - qcopies * NSR * L) % 16 + 16) % 16; /* same bank pair, behind q (and -q) */
          }
          if (L >= 16) addr[g] = e.pos;
          if (L == 1) { /* double coefficient with the q offset in its 16 lowest mantissa bits */
            b[(size_t)m.o_gat + (size_t)(w0 + t) * L + g] =
                (dbits((double)e.coef) & ~0xFFFFull) | (unsigned long long)(e.pos * G * 8);
          } else if (L == CKB_NEGQ_L) { /* coefficient -1: the entry points at -q_s, NSR*L doubles behind q_s (the same bank pair) */
            const int pos = (e.coef < 0 && e.pos < NSR * L) ? e.pos + NSR * L : e.pos;
            b[(size_t)m.o_gat + (size_t)(w0 + t / 4) * L + g] |= (unsigned long long)(pos * G * 8) << (16 * (t & 3));
          } else { /* (sign of the coefficient in bit 31) | offset, two per word */
            const unsigned long long ent = ((e.coef < 0 && e.pos < NSR * L) ? 0x80000000ull : 0ull) | (unsigned long long)(e.pos * G * 8);
            b[(size_t)m.o_gat + (size_t)(w0 + t / 2) * L + g] |= ent << (32 * (t & 1));
          }
        }
        if (L >= 16) out.gather_excess_wavefronts += excess_wavefronts(addr);
        out.gather_steps++;
      }
      w0 += glen[i];
    }
  }
  if (L >= 16) { /* report: excess wavefronts of the concentration reads per f(y) */
    out.slot_excess_wavefronts = 0;
    for (int r = 0; r < NSR; r++)
      for (int k = 0; k < 6; k++) {
        std::vector<int> addr(L, -1);
        for (int g = 0; g < L; g++) {
          const Placed &pl = placed[(size_t)r * L + g];
          addr[g] = k < 3 ? pl.a[k] : pl.b[k - 3];
        }
        out.slot_excess_wavefronts += excess_wavefronts(addr);
      }
  }
  for (int s = 2; s <= s_tab; s++) {
    double mut1;
    std::vector<double> st(4 * (size_t)(s - 1));
    rkc_stage_coefficients(s, &mut1, st.data());
    putd(m.o_rkc + (s - 2), mut1);
    const int base = m.o_rkcs + 4 * ((s - 2) * (s - 1) / 2);
    for (size_t q = 0; q < st.size(); q++) putd(base + (int)q, st[q]);
  }
  return CKB_OK;
}

/* parse once, pack for every lanes-per-system value; the thread-per-ODE packing must fit the kernel
 * parameter space (CKB_PARAM_WORDS) */
int load_packings(const ckb_mech_desc *d, const double *nasa_high, const double *T_mid, const FoDesc *fo, ckb_mech *m) {
  m->parsed = std::make_shared<Parsed>();
  Parsed &P = *m->parsed;
  int rc = parse_mechanism(d, P, fo);
  if (rc != CKB_OK) return rc;
  if ((nasa_high == nullptr) != (T_mid == nullptr)) return CKB_EINVAL;
  if (nasa_high) {
    for (int k = 0; k < P.K; k++) {
      if (!std::isfinite(T_mid[k])) return CKB_EINVAL;
      for (int q = 0; q < 7; q++)
        if (!std::isfinite(nasa_high[7 * (size_t)k + q])) return CKB_EINVAL;
    }
    P.nasa_hi.assign(nasa_high, nasa_high + 7 * (size_t)P.K);
    P.Tmid.assign(T_mid, T_mid + P.K);
  }
  m->K = P.K;
  m->R = P.R;
  m->NS = (int)P.slots.size();
  m->flops_per_rhs = P.flops_per_rhs;
  static const int Ls[CKB_NPACK] = {1, 8, 16, 32, 2, 4};
  bool any = false;
  for (int i = 0; i < CKB_NPACK; i++) {
    Packed &pk = m->pk[i];
    pk.rc = pack_for(P, Ls[i], pk);
    if (pk.rc == CKB_OK && Ls[i] == 1 && pk.dm.words > CKB_PARAM_WORDS) pk.rc = CKB_EUNSUPPORTED;
    if (pk.rc != CKB_OK) pk.blob.clear();
    any = any || pk.rc == CKB_OK;
  }
  if (P.K + 1 > 16) { /* thread-per-ODE beyond the register-resident kernels */
    m->tp.reset(new ThreadPack());
    if (pack_thread(P, *m->tp) != CKB_OK) m->tp.reset();
    any = any || m->tp;
  }
  return any ? CKB_OK : CKB_EUNSUPPORTED;
}

}  // namespace ckb_host

extern "C" int ckb_mech_pack_stats(const ckb_mech_desc *d, int32_t lanes, int32_t *stats8) {
  if (!d || !stats8 || (lanes != 1 && lanes != 2 && lanes != 4 && lanes != 8 && lanes != 16 && lanes != 32)) return CKB_EINVAL;
  ckb_host::Parsed P;
  int rc = ckb_host::parse_mechanism(d, P);
  if (rc != CKB_OK) return rc;
  ckb_host::Packed pk;
  rc = ckb_host::pack_for(P, lanes, pk);
  if (rc != CKB_OK) return rc;
  stats8[0] = pk.dm.NS;
  stats8[1] = pk.dm.NSR;
  stats8[2] = pk.gather_steps;
  stats8[3] = pk.gather_excess_wavefronts;
  stats8[4] = pk.slot_excess_wavefronts;
  stats8[5] = pk.dm.words;
  stats8[6] = ckb::region_doubles(pk.dm);
  stats8[7] = pk.dm.NV;
  return CKB_OK;
}
