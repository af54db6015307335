// trex_host.h -- host-side registry of compiled-in subprocesses and translation of theta[] into kernel parameters.
#pragma once
#include <cmath>
#include <cstdint>

#include "../../include/rex_trex.h"
#include "trex_proc.cuh"

namespace trex {

struct SubprocInfo {
  int npar;        // external legs
  int ncolor;      // colour flows in J^dagger C J
  int nhel;        // helicity combinations summed
  int nunits;      // helicity units a thread block distributes over its warps (antitop helicity closed inside a unit)
  int nvert;       // power of g_s in the amplitude
  double navg;     // spin x colour average x identical-particle factor (R-7)
  int pdg[7];      // process-string order
  QLineLegs qlegs; // light-quark line (quark channels only): row end, column end, gluon, second gluon
};

inline const SubprocInfo* subproc_info(int sid) {
  static SubprocInfo tab[TREX_NSUBPROC];
  static bool ready = false;
  if (!ready) {
    const SubprocInfo base[9] = {
        /* e- e+ > mu- mu+ */ {4, 1, 16, 1, 0, 4.0, {11, -11, 13, -13}, {0, 0, 0}},
        /* g g > t t~      */ {4, 2, 16, 8, 2, 4.0 * 64.0, {21, 21, 6, -6}, {0, 0, 0}},
        /* g g > t t~ g    */ {5, 6, 32, 16, 3, 4.0 * 64.0, {21, 21, 6, -6, 21}, {0, 0, 0}},
        /* g g > t t~ g g  */ {6, 24, 64, 32, 4, 4.0 * 64.0 * 2.0, {21, 21, 6, -6, 21, 21}, {0, 0, 0}},
        /* g g > t t~ g g g*/ {7, 120, 128, 64, 5, 4.0 * 64.0 * 6.0, {21, 21, 6, -6, 21, 21, 21}, {0, 0, 0}},
        /* u u~ > t t~ g   */ {5, 4, 32, 16, 3, 4.0 * 9.0, {2, -2, 6, -6, 21}, {1, 0, 4}},
        /* d d~ > t t~ g   */ {5, 4, 32, 16, 3, 4.0 * 9.0, {1, -1, 6, -6, 21}, {1, 0, 4}},
        /* u g > t t~ u    */ {5, 4, 32, 16, 3, 4.0 * 24.0, {2, 21, 6, -6, 2}, {4, 0, 1}},
        /* g u~ > t t~ u~  */ {5, 4, 32, 16, 3, 4.0 * 24.0, {21, -2, 6, -6, -2}, {1, 4, 0}},
    };
    for (int i = 0; i < 9; ++i) tab[i] = base[i];
    tab[TREX_SP_RESERVED] = SubprocInfo{0, 0, 0, 0, 0, 1.0, {0}, {0, 0, 0}};
    // the other massless flavours: same kernels, another label
    int sid = TREX_SP_SSX_TTG;
    for (int f : {3, 4, 5}) { tab[sid] = base[5]; tab[sid].pdg[0] = f; tab[sid].pdg[1] = -f; ++sid; }
    for (int f : {1, 3, 4, 5}) { tab[sid] = base[7]; tab[sid].pdg[0] = f; tab[sid].pdg[4] = f; ++sid; }
    for (int f : {1, 3, 4, 5}) { tab[sid] = base[8]; tab[sid].pdg[1] = -f; tab[sid].pdg[4] = -f; ++sid; }
    // one light line + two gluons (trex_qq2.cuh): twelve colour flows, 64 helicity combinations of which 32 survive the
    // chirality of the massless line; identical final gluons of q q~ > t t~ g g: 1/2!
    const SubprocInfo two[3] = {
        /* u u~ > t t~ g g  */ {6, 12, 64, 16, 4, 4.0 * 9.0 * 2.0, {2, -2, 6, -6, 21, 21}, {1, 0, 4, 5}},
        /* u g > t t~ u g   */ {6, 12, 64, 16, 4, 4.0 * 24.0, {2, 21, 6, -6, 2, 21}, {4, 0, 1, 5}},
        /* g u~ > t t~ u~ g */ {6, 12, 64, 16, 4, 4.0 * 24.0, {21, -2, 6, -6, -2, 21}, {1, 4, 0, 5}},
    };
    sid = TREX_SP_UUX_TTGG;
    for (int f : {2, 1, 3, 4, 5})
      for (int k = 0; k < 3; ++k) {
        tab[sid] = two[k];
        for (int i = 0; i < 6; ++i) if (tab[sid].pdg[i] == 2 || tab[sid].pdg[i] == -2) tab[sid].pdg[i] = tab[sid].pdg[i] > 0 ? f : -f;
        ++sid;
      }
    ready = true;
  }
  return (sid >= 0 && sid < TREX_NSUBPROC && tab[sid].npar > 0) ? &tab[sid] : nullptr;
}
inline int npar_of_sid(int sid) { const SubprocInfo* sp = subproc_info(sid); return sp ? sp->npar : 0; }
inline bool is_quark_channel(int sid) { return (sid >= TREX_SP_UUX_TTG && sid <= TREX_SP_GUX_TTUX) || (sid >= TREX_SP_SSX_TTG && sid < TREX_NSUBPROC); }
inline bool is_two_gluon_quark_channel(int sid) { return sid >= TREX_SP_UUX_TTGG && sid <= TREX_SP_GBX_TTBXG; }

// returns false if theta is unusable (negative couplings, non-positive scale)
inline bool make_theta_pair(int sid, const double* th_old, const double* th_new, ThetaPair& T) {
  const SubprocInfo* sp = subproc_info(sid);
  if (!sp) return false;
  const double pi = 3.14159265358979323846;
  for (int k = 0; k < 2; ++k) {
    const double* th = k == 0 ? th_old : th_new;
    const double as = th[TREX_TH_ALPHA_S], aem = th[TREX_TH_ALPHA_EM];
    if (sid == TREX_SP_EEMUMU) {
      const double sw2 = th[TREX_TH_SIN2W];
      if (!(aem >= 0.0) || !(sw2 > 0.0) || !(sw2 < 1.0)) return false;
      const double e2 = 4.0 * pi * aem, e = std::sqrt(e2), sc = std::sqrt(sw2 * (1.0 - sw2));
      T.e2[k] = e2; T.gL[k] = e / sc * (-0.5 + sw2); T.gR[k] = e / sc * sw2;
      T.mZ2[k] = th[TREX_TH_MZ] * th[TREX_TH_MZ]; T.mZGZ[k] = th[TREX_TH_MZ] * th[TREX_TH_GAMMAZ];
      T.mt[k] = T.mGt[k] = T.kq[k] = 0.0;
      T.pref[k] = 1.0 / sp->navg; T.gs2nv[k] = 1.0;
    } else {
      if (!(as >= 0.0) || !(th[TREX_TH_LAMBDA] > 0.0)) return false;
      const double gs = std::sqrt(4.0 * pi * as);
      const double kappa = th[TREX_TH_CTG] * th[TREX_TH_VEV] / (std::sqrt(2.0) * th[TREX_TH_LAMBDA] * th[TREX_TH_LAMBDA]);
      T.mt[k] = th[TREX_TH_MT]; T.mGt[k] = th[TREX_TH_MT] * th[TREX_TH_GAMMAT];
      if (!std::isfinite(kappa) || !std::isfinite(th[TREX_TH_MT]) || !std::isfinite(th[TREX_TH_GAMMAT])) return false;
      T.kq[k] = gs > 0.0 ? kappa / gs : 0.0;      // alpha_s = 0: pref = 0, so |M|^2 = 0 exactly (zero guard applies)
      T.pref[k] = std::pow(gs, 2 * sp->nvert) / sp->navg; T.gs2nv[k] = std::pow(gs, 2 * sp->nvert);
      T.e2[k] = T.gL[k] = T.gR[k] = T.mZ2[k] = T.mZGZ[k] = 0.0;
    }
  }
  return true;
}

}  // namespace trex
