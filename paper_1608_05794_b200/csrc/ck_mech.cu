// Mechanism packer: validates a ck_mech_desc, regroups reactions by type, folds the equilibrium
// constant into a per-interval polynomial for ln k_r, builds the SoA arrays and uploads them.
//
// Reverse rate (Eq. 16-18) with the NASA-7 forms of Eq. 19:
//   ln k_r = ln k_f - ln K_c,  ln K_c = dnu ln(p0/(R_u T)) - sum_k nu_ki g_k,
//   g_k = H_k/(R T) - S_k/R = (a1 - a7) - a1 lnT - a2 T/2 - a3 T^2/6 - a4 T^3/12 - a5 T^4/20 + a6/T
// so, with DA_j = sum_k nu_ki a_jk over the NASA range each species is in,
//   ln k_r = [lnA - dnu ln(p0/R_u) + DA_1 - DA_7] + [beta + dnu - DA_1] lnT + [DA_6 - Ta]/T
//            - DA_2/2 T - DA_3/6 T^2 - DA_4/12 T^3 - DA_5/20 T^4 .
// The range of a species switches at its own t_mid, so the coefficients are tabulated per temperature
// interval between consecutive distinct t_mid values (one interval pair for GRI-style models).
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>

#include "ck_internal.h"

namespace ck {

static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
}
int32_t cuda_fail(cudaError_t e, const char* what) {
  set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
  return CK_ECUDA;
}

namespace {
struct Arena {
  std::vector<unsigned char> buf;
  template <class T>
  size_t put(const std::vector<T>& v) {
    size_t off = (buf.size() + 255) & ~size_t(255);
    size_t bytes = std::max<size_t>(v.size() * sizeof(T), 8);
    buf.resize(off + bytes, 0);
    if (!v.empty()) std::memcpy(buf.data() + off, v.data(), v.size() * sizeof(T));
    return off;
  }
};
}  // namespace
}  // namespace ck

using namespace ck;

extern "C" const char* ck_last_error(void) { return ck::g_err; }
extern "C" int32_t ck_version(void) { return 100; }

extern "C" int32_t ck_mech_load(const ck_mech_desc* d, int32_t device, ck_mech** out) {
  if (!d || !out) { set_error("ck_mech_load: null argument"); return CK_EINVAL; }
  *out = nullptr;
  if (d->struct_size != (int32_t)sizeof(ck_mech_desc)) { set_error("ck_mech_load: struct_size mismatch"); return CK_EINVAL; }
  const int K = d->n_species, R = d->n_reactions, E = d->n_elements;
  if (K < 1 || R < 0 || K > 8000000) { set_error("ck_mech_load: bad sizes K=%d R=%d", K, R); return CK_EINVAL; }
  if (!d->mol_wt || !d->nasa_lo || !d->nasa_hi || !d->t_mid) { set_error("ck_mech_load: null species arrays"); return CK_EINVAL; }
  if (R > 0 && (!d->reac_ptr || !d->prod_ptr || !d->reac_spec || !d->reac_nu || !d->prod_spec || !d->prod_nu || !d->A ||
                !d->beta || !d->Ea || !d->reversible || !d->type)) {
    set_error("ck_mech_load: null reaction arrays"); return CK_EINVAL;
  }
  for (int k = 0; k < K; ++k)
    if (!(d->mol_wt[k] > 0) || !std::isfinite(d->mol_wt[k])) { set_error("ck_mech_load: mol_wt[%d] not positive", k); return CK_EINVAL; }

  // ---- temperature intervals ---------------------------------------------------------------------
  std::vector<double> edges(d->t_mid, d->t_mid + K);
  std::sort(edges.begin(), edges.end());
  edges.erase(std::unique(edges.begin(), edges.end()), edges.end());
  const int nT = (int)edges.size() + 1;
  if (nT > MAX_TINT) { set_error("ck_mech_load: %d distinct t_mid values (max %d)", nT - 1, MAX_TINT - 1); return CK_EUNSUPPORTED; }

  // ---- regroup reactions by type (plain rows: those with six distinct slot species first) ------------
  auto has_dup = [&](int i) {
    for (int x = d->reac_ptr[i]; x < d->reac_ptr[i + 1]; ++x) {
      if (d->reac_nu[x] != 1) return true;
      for (int x2 = d->reac_ptr[i]; x2 < x; ++x2)
        if (d->reac_spec[x2] == d->reac_spec[x]) return true;
      for (int y = d->prod_ptr[i]; y < d->prod_ptr[i + 1]; ++y)
        if (d->prod_spec[y] == d->reac_spec[x]) return true;
    }
    for (int y = d->prod_ptr[i]; y < d->prod_ptr[i + 1]; ++y) {
      if (d->prod_nu[y] != 1) return true;
      for (int y2 = d->prod_ptr[i]; y2 < y; ++y2)
        if (d->prod_spec[y2] == d->prod_spec[y]) return true;
    }
    return false;
  };
  std::vector<int> perm;
  int cnt[4] = {0, 0, 0, 0};
  int r_dup = 0;
  for (int i = 0; i < R; ++i) {
    if (d->type[i] > 3) { set_error("ck_mech_load: type[%d]=%d", i, (int)d->type[i]); return CK_EINVAL; }
    if (d->reac_ptr[i + 1] < d->reac_ptr[i] || d->prod_ptr[i + 1] < d->prod_ptr[i]) { set_error("ck_mech_load: CSR pointers of reaction %d decrease", i); return CK_EINVAL; }
  }
  // A row may join the fast groups only if the arguments of BOTH of its exponentials stay inside (-680, 680) for
  // every temperature in [T_SAFE_LO, T_SAFE_HI]: the kernels then evaluate them without range checks whenever
  // all 32 reactors of a warp are inside that temperature window (ck_exp_nc, ck_chem.cuh).
  auto bounded = [&](int i) {
    if (!d->reversible[i] || !(d->A[i] > 0)) return false;
    std::map<int, int> net;
    int dnu = 0;
    for (int x = d->reac_ptr[i]; x < d->reac_ptr[i + 1]; ++x) {
      if (d->reac_spec[x] < 0 || d->reac_spec[x] >= K) return false;
      net[d->reac_spec[x]] -= d->reac_nu[x]; dnu -= d->reac_nu[x];
    }
    for (int x = d->prod_ptr[i]; x < d->prod_ptr[i + 1]; ++x) {
      if (d->prod_spec[x] < 0 || d->prod_spec[x] >= K) return false;
      net[d->prod_spec[x]] += d->prod_nu[x]; dnu += d->prod_nu[x];
    }
    const double lnA_ = std::log(d->A[i]), Ta_ = d->Ea[i] / R_CAL;
    for (int sidx = 0; sidx <= 256; ++sidx) {
      const double T = T_SAFE_LO * std::pow(T_SAFE_HI / T_SAFE_LO, sidx / 256.0), lnT = std::log(T);
      const double xf = lnA_ + d->beta[i] * lnT - Ta_ / T;
      double sum = 0;
      for (auto& kv : net) {
        const int k = kv.first;
        const double* a = (T > d->t_mid[k]) ? &d->nasa_hi[7 * k] : &d->nasa_lo[7 * k];
        const double g = a[0] * (1 - lnT) - a[1] * T / 2 - a[2] * T * T / 6 - a[3] * T * T * T / 12 - a[4] * T * T * T * T / 20 +
                         a[5] / T - a[6];
        sum += kv.second * g;
      }
      const double xr = xf - (dnu * std::log(P_0 / (R_U * T)) - sum);
      if (!(std::fabs(xf) < 680.0) || !(std::fabs(xr) < 680.0)) return false;
    }
    return true;
  };
  std::vector<char> slow(R, 0);
  for (int i = 0; i < R; ++i) slow[i] = (d->type[i] != 0) || has_dup(i) || !bounded(i);
  // at most two reactants and two products (all distinct, nu = 1): slots 0, 1, 3, 4 only; a missing partner is the
  // dummy species K (C[K] = 1, accumulator column K is a sink), so the group runs without predicates
  auto is22 = [&](int i) { return d->reac_ptr[i + 1] - d->reac_ptr[i] <= 2 && d->prod_ptr[i + 1] - d->prod_ptr[i] <= 2; };
  int r_22 = 0;
  for (int i = 0; i < R; ++i) if (!slow[i] && is22(i)) { perm.push_back(i); cnt[0]++; r_dup++; r_22++; }
  for (int i = 0; i < R; ++i) if (!slow[i] && !is22(i)) { perm.push_back(i); cnt[0]++; r_dup++; }
  for (int i = 0; i < R; ++i) if (d->type[i] == 0 && slow[i]) { perm.push_back(i); cnt[0]++; }
  int n_tbf = 0;  // three-body rows that qualify for the fast path come first in their group
  auto tb_fast = [&](int i) {
    return d->type[i] == 1 && d->eff_ptr && !has_dup(i) && bounded(i) && d->eff_ptr[i + 1] - d->eff_ptr[i] <= 6 &&
           d->eff_ptr[i + 1] >= d->eff_ptr[i];
  };
  for (int i = 0; i < R; ++i) if (tb_fast(i)) { perm.push_back(i); cnt[1]++; n_tbf++; }
  for (int i = 0; i < R; ++i) if (d->type[i] == 1 && !tb_fast(i)) { perm.push_back(i); cnt[1]++; }
  for (int t = 2; t < 4; ++t)
    for (int i = 0; i < R; ++i)
      if (d->type[i] == t) { perm.push_back(i); cnt[t]++; }
  const int r_tb = cnt[0], r_lind = cnt[0] + cnt[1], r_troe = r_lind + cnt[2];
  if (cnt[1] + cnt[2] + cnt[3] > 0 && (!d->eff_ptr)) { set_error("ck_mech_load: eff_ptr missing"); return CK_EINVAL; }
  if (cnt[2] + cnt[3] > 0 && (!d->A0 || !d->beta0 || !d->Ea0)) { set_error("ck_mech_load: low-pressure arrays missing"); return CK_EINVAL; }
  if (cnt[3] > 0 && !d->troe) { set_error("ck_mech_load: troe missing"); return CK_EINVAL; }

  std::vector<double> W(d->mol_wt, d->mol_wt + K), invW(K), nlo(7 * K), nhi(7 * K), tmid(d->t_mid, d->t_mid + K);
  for (int k = 0; k < K; ++k) {
    invW[k] = 1.0 / W[k];
    for (int j = 0; j < 7; ++j) { nlo[j * K + k] = d->nasa_lo[7 * k + j]; nhi[j * K + k] = d->nasa_hi[7 * k + j]; }
  }
  std::vector<double> lnA(R), beta(R), Ta(R), krc((size_t)nT * 7 * R);
  std::vector<int> slot(6 * (size_t)std::max(R, 1), K);
  std::vector<int> eptr(1, 0), espec;
  std::vector<double> eval1;
  std::vector<double> lnA0, beta0, Ta0, troe(4 * (size_t)std::max(cnt[3], 1), 0.0);
  std::vector<std::vector<std::pair<int, int>>> tr(K);  // species -> (reaction, net nu)
  long long n_part = 0;
  int n_rev = 0;

  for (int r = 0; r < R; ++r) {
    const int i = perm[r];
    if (!(d->A[i] > 0) || !std::isfinite(d->A[i])) { set_error("ck_mech_load: A[%d] not positive", i); return CK_EINVAL; }
    lnA[r] = std::log(d->A[i]); beta[r] = d->beta[i]; Ta[r] = d->Ea[i] / R_CAL;
    std::map<int, int> net;
    std::vector<long long> bal(std::max(E, 1), 0);
    for (int side = 0; side < 2; ++side) {
      const int32_t* ptr = side ? d->prod_ptr : d->reac_ptr;
      const int32_t* sp = side ? d->prod_spec : d->reac_spec;
      const int32_t* nu = side ? d->prod_nu : d->reac_nu;
      const int b = ptr[i], e = ptr[i + 1];
      if (e < b) { set_error("ck_mech_load: CSR pointers of reaction %d decrease", i); return CK_EINVAL; }
      int filled = 0;
      for (int x = b; x < e; ++x) {
        if (sp[x] < 0 || sp[x] >= K || nu[x] < 1 || nu[x] > 3) { set_error("ck_mech_load: reaction %d: bad species/nu", i); return (nu[x] > 3) ? CK_EUNSUPPORTED : CK_EINVAL; }
        for (int y = b; y < x; ++y)
          if (sp[y] == sp[x]) { set_error("ck_mech_load: reaction %d lists species %d twice on one side", i, sp[x]); return CK_EINVAL; }
        for (int c = 0; c < nu[x]; ++c) {
          if (filled == 3) { set_error("ck_mech_load: reaction %d has molecularity > 3 on one side", i); return CK_EUNSUPPORTED; }
          slot[(size_t)(side * 3 + filled) * R + r] = sp[x];
          filled++;
        }
        net[sp[x]] += side ? nu[x] : -nu[x];
        if (d->elem_comp) for (int el = 0; el < E; ++el) bal[el] += (side ? 1 : -1) * (long long)nu[x] * d->elem_comp[(size_t)sp[x] * E + el];
        n_part += nu[x];
      }
    }
    if (d->elem_comp)
      for (int el = 0; el < E; ++el)
        if (bal[el] != 0) { set_error("ck_mech_load: reaction %d does not balance element %d", i, el); return CK_EINVAL; }
    int dnu = 0;
    for (auto& kv : net) { dnu += kv.second; if (kv.second != 0) tr[kv.first].push_back({r, kv.second}); }
    // ln k_r polynomial per interval (long double accumulation of the coefficient sums)
    for (int t = 0; t < nT; ++t) {
      double* c = &krc[((size_t)t * 7) * R + r];
      if (!d->reversible[i]) {
        c[0] = -std::numeric_limits<double>::infinity();
        for (int j = 1; j < 7; ++j) c[(size_t)j * R] = 0.0;
        continue;
      }
      long double DA[7] = {0, 0, 0, 0, 0, 0, 0};
      for (auto& kv : net) {
        const int k = kv.first;
        // interval t lies above t_mid[k] iff its lower edge edges[t-1] >= t_mid[k]
        const bool high = (t > 0) && (edges[t - 1] >= d->t_mid[k]);
        const double* a = high ? &d->nasa_hi[7 * k] : &d->nasa_lo[7 * k];
        for (int j = 0; j < 7; ++j) DA[j] += (long double)kv.second * a[j];
      }
      c[0] = (double)((long double)lnA[r] - dnu * std::log((long double)P_0 / R_U) + DA[0] - DA[6]);
      c[(size_t)1 * R] = (double)((long double)beta[r] + dnu - DA[0]);
      c[(size_t)2 * R] = (double)(DA[5] - (long double)Ta[r]);
      c[(size_t)3 * R] = (double)(-DA[1] / 2);
      c[(size_t)4 * R] = (double)(-DA[2] / 6);
      c[(size_t)5 * R] = (double)(-DA[3] / 12);
      c[(size_t)6 * R] = (double)(-DA[4] / 20);
    }
    if (d->reversible[i]) n_rev++;
    if (r >= r_tb) {
      for (int x = d->eff_ptr[i]; x < d->eff_ptr[i + 1]; ++x) {
        if (d->eff_spec[x] < 0 || d->eff_spec[x] >= K) { set_error("ck_mech_load: reaction %d: bad efficiency species", i); return CK_EINVAL; }
        espec.push_back(d->eff_spec[x]); eval1.push_back(d->eff_val[x] - 1.0);
      }
      eptr.push_back((int)espec.size());
    }
    if (r >= r_lind) {
      if (!(d->A0[i] > 0)) { set_error("ck_mech_load: A0[%d] not positive", i); return CK_EINVAL; }
      lnA0.push_back(std::log(d->A0[i])); beta0.push_back(d->beta0[i]); Ta0.push_back(d->Ea0[i] / R_CAL);
    }
    if (r >= r_troe) {
      const int j = r - r_troe, nt = cnt[3];
      const double* tp = &d->troe[4 * (size_t)i];
      if (tp[1] == 0 || tp[2] == 0) { set_error("ck_mech_load: Troe T*** / T* of reaction %d is zero", i); return CK_EINVAL; }
      troe[j] = tp[0]; troe[nt + j] = 1.0 / tp[1]; troe[2 * nt + j] = 1.0 / tp[2]; troe[3 * nt + j] = tp[3];
    }
  }
  if (K > 1022) { set_error("ck_mech_load: more than 1022 species"); return CK_EUNSUPPORTED; }
  const int rstride = RPH + 8 * nT;
  std::vector<double> rpack((size_t)std::max(R, 1) * rstride, 0.0);
  std::vector<int> rflag(std::max(R, 1), 0);
  for (int r = 0; r < R; ++r) {
    double* q = &rpack[(size_t)r * rstride];
    q[0] = lnA[r]; q[1] = beta[r]; q[2] = Ta[r];
    uint32_t w[2] = {0, 0};
    for (int s = 0; s < 6; ++s) w[s / 3] |= (uint32_t)slot[(size_t)s * R + r] << (10 * (s % 3));
    bool dup = false;  // a species in two slots: the omega scatter of this row must run slot by slot
    for (int s = 0; s < 6; ++s)
      for (int s2 = 0; s2 < s; ++s2)
        if (slot[(size_t)s * R + r] != K && slot[(size_t)s * R + r] == slot[(size_t)s2 * R + r]) dup = true;
    if (dup) { w[1] |= 0x80000000u; rflag[r] = 1; }
    std::memcpy(&q[3], w, sizeof w);
    const uint32_t pre[4] = {(uint32_t)slot[(size_t)0 * R + r] << 12, (uint32_t)slot[(size_t)1 * R + r] << 12,
                             (uint32_t)slot[(size_t)3 * R + r] << 12, (uint32_t)slot[(size_t)4 * R + r] << 12};
    std::memcpy(&q[4], pre, sizeof pre);
    for (int t = 0; t < nT; ++t)
      for (int j = 0; j < 7; ++j) q[RPH + 8 * t + j] = krc[((size_t)t * 7 + j) * R + r];
  }
  const int n_special = R - r_tb;
  std::vector<double> xpack((size_t)std::max(n_special, 1) * 16, 0.0);
  for (int j = 0; j < n_special; ++j) {
    double* q = &xpack[(size_t)j * 16];
    const int r = r_tb + j;
    if (r >= r_lind) { q[0] = lnA0[r - r_lind]; q[1] = beta0[r - r_lind]; q[2] = Ta0[r - r_lind]; }
    if (r >= r_troe) { const int jt = r - r_troe, nt = cnt[3]; q[3] = troe[jt]; q[4] = troe[nt + jt]; q[5] = troe[2 * nt + jt]; q[6] = troe[3 * nt + jt]; }
    const int e0 = eptr[j], ne = eptr[j + 1] - e0;
    uint64_t w = (ne <= 6) ? (uint64_t)ne : 15u;
    if (ne <= 6)
      for (int x = 0; x < ne; ++x) { w |= (uint64_t)espec[e0 + x] << (4 + 10 * x); q[8 + x] = eval1[e0 + x]; }
    std::memcpy(&q[7], &w, sizeof w);
  }
  std::vector<double> spack((size_t)K * SPS, 0.0);
  for (int k = 0; k < K; ++k) {
    double* q = &spack[(size_t)k * SPS];
    q[0] = W[k]; q[1] = invW[k]; q[2] = tmid[k];
    const double hs[5] = {1.0, 0.5, 1.0 / 3.0, 0.25, 0.2};
    for (int rg = 0; rg < 2; ++rg) {
      const double* a = rg ? &d->nasa_hi[7 * k] : &d->nasa_lo[7 * k];
      for (int j = 0; j < 5; ++j) { q[4 + 5 * rg + j] = a[j]; q[14 + 6 * rg + j] = a[j] * hs[j]; }
      q[14 + 6 * rg + 5] = a[5];
    }
  }
  std::vector<int> tptr(K + 1, 0), tent;
  for (int k = 0; k < K; ++k) {
    for (auto& pr : tr[k]) tent.push_back((pr.first << 8) | (pr.second + 128));
    tptr[k + 1] = (int)tent.size();
  }

  // ---- arena + upload -------------------------------------------------------------------------------
  Arena a;
  size_t oW = a.put(W), oiW = a.put(invW), olo = a.put(nlo), ohi = a.put(nhi), otm = a.put(tmid);
  size_t olnA = a.put(lnA), ob = a.put(beta), oTa = a.put(Ta), okrc = a.put(krc), oslot = a.put(slot), osp = a.put(spack), oxp = a.put(xpack), orf = a.put(rflag);
  size_t oep = a.put(eptr), oes = a.put(espec), oev = a.put(eval1);
  size_t olnA0 = a.put(lnA0), ob0 = a.put(beta0), oTa0 = a.put(Ta0), otroe = a.put(troe);
  size_t otp = a.put(tptr), ote = a.put(tent), operm = a.put(perm), orp = a.put(rpack);

  ck_mech* m = new ck_mech;
  m->device = device;
  cudaError_t e = cudaSetDevice(device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&m->sms, cudaDevAttrMultiProcessorCount, device);
  if (e == cudaSuccess) e = cudaMalloc(&m->arena, a.buf.size());
  if (e == cudaSuccess) e = cudaMemcpy(m->arena, a.buf.data(), a.buf.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    if (m->arena) cudaFree(m->arena);
    delete m;
    return cuda_fail(e, "ck_mech_load upload");
  }
  m->arena_bytes = a.buf.size();
  const char* base = (const char*)m->arena;
  MechDev& v = m->dev;
  v.K = K; v.R = R; v.nT = nT; v.cv = 0;
  v.t_safe_lo = T_SAFE_LO; v.t_safe_hi = T_SAFE_HI;
  v.r_tbf = r_tb + n_tbf;
  v.r_22 = r_22; v.r_dup = r_dup; v.r_tb = r_tb; v.r_lind = r_lind; v.r_troe = r_troe;
  for (int t = 0; t < MAX_TINT; ++t) v.tedge[t] = (t < nT - 1) ? edges[t] : std::numeric_limits<double>::infinity();
  v.W = (const double*)(base + oW); v.invW = (const double*)(base + oiW);
  v.nlo = (const double*)(base + olo); v.nhi = (const double*)(base + ohi); v.tmid = (const double*)(base + otm);
  v.lnA = (const double*)(base + olnA); v.beta = (const double*)(base + ob); v.Ta = (const double*)(base + oTa);
  v.krc = (const double*)(base + okrc); v.slot = (const int*)(base + oslot); v.spack = (const double*)(base + osp); v.xpack = (const double*)(base + oxp); v.rflag = (const int*)(base + orf);
  v.eptr = (const int*)(base + oep); v.espec = (const int*)(base + oes); v.eval1 = (const double*)(base + oev);
  v.lnA0 = (const double*)(base + olnA0); v.beta0 = (const double*)(base + ob0); v.Ta0 = (const double*)(base + oTa0);
  v.troe = (const double*)(base + otroe);
  v.rpack = (const double*)(base + orp); v.rstride = rstride;
  v.tptr = (const int*)(base + otp); v.tent = (const int*)(base + ote); v.n_tent = (int)tent.size(); v.perm = (const int*)(base + operm);
  m->K = K; m->R = R; m->n_tb = cnt[1]; m->n_lind = cnt[2]; m->n_troe = cnt[3]; m->n_rev = n_rev;
  m->n_part = n_part; m->n_eff = (long long)espec.size();
  *out = m;
  return CK_OK;
}

extern "C" int32_t ck_mech_free(ck_mech* m) {
  if (!m) return CK_OK;
  cudaSetDevice(m->device);
  if (m->arena) cudaFree(m->arena);
  if (m->stage) cudaFree(m->stage);
  if (m->hstream) cudaStreamDestroy(m->hstream);
  for (auto& ps : m->pstream) if (ps) cudaStreamDestroy(ps);
  delete m;
  return CK_OK;
}

extern "C" int32_t ck_mech_set_reactor(ck_mech* m, int32_t kind) {
  if (!m || (kind != CK_CONST_PRESSURE && kind != CK_CONST_VOLUME)) { set_error("ck_mech_set_reactor: bad argument"); return CK_EINVAL; }
  m->dev.cv = (kind == CK_CONST_VOLUME) ? 1 : 0;
  return CK_OK;
}

extern "C" int32_t ck_mech_sizes(const ck_mech* m, int32_t* n_species, int32_t* n_reactions) {
  if (!m) { set_error("ck_mech_sizes: null handle"); return CK_EINVAL; }
  if (n_species) *n_species = m->K;
  if (n_reactions) *n_reactions = m->R;
  return CK_OK;
}

// Algorithmic FP64 "slots" of one RHS evaluation: transcendental
// functions at their sm_100a FP64-pipe instruction counts (exp 15, log 29, div 8), FMA/MUL/ADD 1.
extern "C" int32_t ck_rhs_slots(const ck_mech* m, double* slots) {
  if (!m || !slots) { set_error("ck_rhs_slots: null argument"); return CK_EINVAL; }
  const double EXP = 15, LOG = 29, DIV = 8;
  double s = LOG + DIV + 6;                         // lnT, 1/T, powers of T
  s += m->K * (2.0 /*S*/ + 2.0 /*C_k*/ + 6.0 /*cp/R + cp sum*/ + 7.0 /*H/RT*/ + 2.0 /*hw*/ + 2.0 /*Ydot*/);
  s += 2 * DIV + 6;                                 // rho, 1/rho, Tdot
  s += m->R * (3.0 + EXP);                          // k_f
  s += m->n_rev * (7.0 + EXP);                      // k_r polynomial + exp
  s += (double)m->n_part * 1.0 + m->R * 3.0;        // concentration products, q
  s += (double)m->n_part * 1.0;                     // omega scatter
  s += (m->n_tb + m->n_lind + m->n_troe) * 1.0 + (double)m->n_eff; // [M]
  s += (m->n_lind + m->n_troe) * (3.0 + EXP + 2.0 + 2 * DIV);       // k_0, Pr, Pr/(1+Pr)
  s += m->n_troe * (3 * EXP + 5.0 + 2 * LOG + 2.0 + 8.0 + 2 * DIV + EXP); // F_cent, logs, f1, F
  *slots = s;
  return CK_OK;
}
