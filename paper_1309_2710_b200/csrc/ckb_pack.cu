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

struct Rx {
  std::vector<int> reac, prod; /* molecule lists (species repeated nu times), sorted */
  int tbset = -1;
};

}  // namespace

struct Parsed {
  int K = 0, R = 0;
  std::vector<double> W, nasa;                                  /* [K], [K][7] */
  std::vector<double> A, beta, E;                               /* [R] */
  std::vector<Rx> rx;                                           /* [R] */
  std::vector<std::vector<std::pair<int, double>>> sets;        /* third-body sets: (species, alpha) */
  struct Slot { int f, r; };
  std::vector<Slot> slots;                                      /* fused forward/reverse pairs */
  std::vector<std::vector<std::pair<int, int>>> rows;           /* [K] gather rows: (slot, net coefficient) */
  double flops_per_rhs = 0.0;
};

int parse_mechanism(const ckb_mech_desc *d, Parsed &P) {
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
  if (P.sets.size() > 65000) return CKB_EUNSUPPORTED;

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
  P.flops_per_rhs = F;
  return CKB_OK;
}

/* RKC coefficients of an s-stage step, Eq. 22-26 with R8 (w0 = 1 + (2/13)/s^2), R9
 * (a_j = 1 - b_j T_j(w0)) and R10 (b_0 = b_1 = b_2).  out: mu~_1, then (mu_j, nu_j, mu~_j, gamma~_j), j = 2..s. */
static void rkc_coefficients(int s, double *mut1, double *stages) {
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

int pack_for(const Parsed &P, int L, Packed &out) {
  const int K = P.K, n = K + 1, G = 32 / L;
  const int NS = (int)P.slots.size(), NTB = (int)P.sets.size();
  const int NV = pick_nv(L, n), NSR = (NS + L - 1) / L, NTBR = (NTB + L - 1) / L;
  if (NV < 0) return CKB_EUNSUPPORTED;
  int TBE = 0;
  for (auto &s : P.sets) TBE = std::max(TBE, (int)s.size());
  /* 16-bit region offsets */
  if ((long long)(n + NTB) * G > 65535 || (long long)NSR * L * G > 65535) return CKB_EUNSUPPORTED;

  /* components: 0 = T, then species by decreasing gather-row length */
  std::vector<int> sp_of_comp(n, -1), comp_of_sp(K);
  {
    std::vector<int> order(K);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(),
                     [&](int a, int b) { return P.rows[a].size() > P.rows[b].size(); });
    for (int c = 1; c < n; c++) {
      sp_of_comp[c] = order[c - 1];
      comp_of_sp[order[c - 1]] = c;
    }
  }
  std::vector<int> glen(NV, 0);
  for (int c = 1; c < n; c++) glen[c / L] = std::max(glen[c / L], (int)P.rows[sp_of_comp[c]].size());
  const int gsteps = std::accumulate(glen.begin(), glen.end(), 0);
  const int s_tab = (L == 1) ? 12 : 48;

  ckb::DevMech &m = out.dm;
  m.K = K; m.n = n; m.L = L; m.NV = NV; m.NS = NS; m.NSR = NSR; m.NTB = NTB; m.NTBR = NTBR; m.TBE = TBE;
  int off = 0;
  auto take = [&off](size_t words) { int o = off; off += (int)words; return o; };
  m.o_sp = take((size_t)NV * CKB_SP_WORDS * L);
  m.o_sl = take((size_t)NSR * CKB_SL_WORDS * L);
  m.o_tb = take((size_t)NTBR * TBE * 2 * L);
  m.o_glen = take(NV);
  m.o_gat = take((size_t)gsteps * L);
  m.o_perm = take(n);
  m.s_tab = s_tab;
  m.o_rkc = take(s_tab - 1);
  m.o_rkcs = take((size_t)4 * (s_tab - 1) * s_tab / 2);
  m.words = off;
  std::vector<unsigned long long> &b = out.blob;
  b.assign((size_t)off, 0ull);
  auto putd = [&b](int o, double x) { b[(size_t)o] = dbits(x); };

  for (int c = 0; c < NV * L; c++) { /* species table; T and padding components keep zeros (W = 1) */
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
  for (int c = 0; c < n; c++) b[(size_t)m.o_perm + c] = (unsigned long long)(c == 0 ? 0 : 1 + sp_of_comp[c]);

  const double NEG_INF = -1.0e4; /* stands for ln 0: ckb_exp() returns ~1e-308 for it, no special case on the device */
  for (int s = 0; s < NSR * L; s++) {
    const int r = s / L, g = s % L, base = m.o_sl + r * CKB_SL_WORDS * L + g;
    unsigned long long wa = 0, wb = 0;
    if (s < NS) {
      const int f = P.slots[s].f, rv = P.slots[s].r;
      putd(base + CKB_SL_LNAF * L, P.A[f] > 0.0 ? std::log(P.A[f]) : NEG_INF);
      putd(base + CKB_SL_BF * L, P.beta[f]);
      putd(base + CKB_SL_THF * L, P.E[f] / RC_CAL);
      putd(base + CKB_SL_LNAR * L, (rv >= 0 && P.A[rv] > 0.0) ? std::log(P.A[rv]) : NEG_INF);
      putd(base + CKB_SL_BR * L, rv >= 0 ? P.beta[rv] : 0.0);
      putd(base + CKB_SL_THR * L, rv >= 0 ? P.E[rv] / RC_CAL : 0.0);
      const Rx &x = P.rx[f];
      for (int q = 0; q < 3; q++) {
        /* absent molecule -> C_0 = 1; a slot without reverse multiplies k_r = 0 by 1, never by a concentration */
        const unsigned long long ao = q < (int)x.reac.size() ? (unsigned)(comp_of_sp[x.reac[q]] * G) : 0u;
        const unsigned long long bo = (rv >= 0 && q < (int)x.prod.size()) ? (unsigned)(comp_of_sp[x.prod[q]] * G) : 0u;
        wa |= ao << (16 * q);
        wb |= bo << (16 * q);
      }
      wa |= (unsigned long long)((n + (x.tbset >= 0 ? x.tbset : NTB)) * G) << 48;
    } else { /* padding slot: q = 0 */
      putd(base + CKB_SL_LNAF * L, NEG_INF);
      putd(base + CKB_SL_LNAR * L, NEG_INF);
      wa = (unsigned long long)((n + NTB) * G) << 48;
    }
    b[(size_t)base + CKB_SL_IDXA * L] = wa;
    b[(size_t)base + CKB_SL_IDXB * L] = wb;
  }
  for (int t = 0; t < NTBR * L; t++) { /* third-body sets, padded with (alpha - 1) = 0 on C_0 */
    const int r = t / L, g = t % L;
    for (int e = 0; e < TBE; e++) {
      const int base = m.o_tb + ((r * TBE + e) * 2) * L + g;
      if (t < NTB && e < (int)P.sets[t].size()) {
        putd(base, P.sets[t][e].second - 1.0);
        b[(size_t)base + L] = (unsigned long long)(comp_of_sp[P.sets[t][e].first] * G);
      }
    }
  }
  {
    int step0 = 0;
    for (int i = 0; i < NV; i++) {
      b[(size_t)m.o_glen + i] = (unsigned long long)glen[i];
      for (int g = 0; g < L; g++) {
        const int c = g + L * i;
        if (c < 1 || c >= n) continue;
        const auto &row = P.rows[sp_of_comp[c]];
        for (int t = 0; t < (int)row.size(); t++)
          b[(size_t)m.o_gat + (size_t)(step0 + t) * L + g] =
              (dbits((double)row[t].second) & ~0xFFFFull) | (unsigned long long)(row[t].first * G);
      }
      step0 += glen[i];
    }
  }
  for (int s = 2; s <= s_tab; s++) {
    double mut1;
    std::vector<double> st(4 * (size_t)(s - 1));
    rkc_coefficients(s, &mut1, st.data());
    putd(m.o_rkc + (s - 2), mut1);
    const int base = m.o_rkcs + 4 * ((s - 2) * (s - 1) / 2);
    for (size_t q = 0; q < st.size(); q++) putd(base + (int)q, st[q]);
  }
  return CKB_OK;
}


/* parse once, pack for every lanes-per-system value; the thread-per-ODE packing must fit the kernel
 * parameter space (CKB_PARAM_WORDS) */
int load_packings(const ckb_mech_desc *d, ckb_mech *m) {
  Parsed P;
  int rc = parse_mechanism(d, P);
  if (rc != CKB_OK) return rc;
  m->K = P.K;
  m->R = P.R;
  m->NS = (int)P.slots.size();
  m->flops_per_rhs = P.flops_per_rhs;
  static const int Ls[4] = {1, 8, 16, 32};
  bool any = false;
  for (int i = 0; i < 4; i++) {
    Packed &pk = m->pk[i];
    pk.rc = pack_for(P, Ls[i], pk);
    if (pk.rc == CKB_OK && Ls[i] == 1 && pk.dm.words > CKB_PARAM_WORDS) pk.rc = CKB_EUNSUPPORTED;
    if (pk.rc != CKB_OK) pk.blob.clear();
    any = any || pk.rc == CKB_OK;
  }
  return any ? CKB_OK : CKB_EUNSUPPORTED;
}

}  // namespace ckb_host
