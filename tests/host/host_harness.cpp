// TEST-ONLY harness: runs the GENERATED matrix-element programs (csrc/generated/*.inc, csrc/helas.cuh,
// csrc/me_tasks.cuh) on the CPU by emulating the lanes of a warp one after the other.  It exists so the
// generator's diagram / colour / phase logic and the vertex routines can be checked against the oracle in the
// `-m "not gpu"` suite, where no GPU is available.  It is compiled by tests/test_generated_host.py with g++ and
// is NOT part of the product library: libmadme.so has no CPU path.
#include <cmath>
#include <cstring>
#include <vector>
#include "../../paper_2211_14056_b200/csrc/generated/epem_mupmum.inc"
#include "../../paper_2211_14056_b200/csrc/generated/gg_ttx.inc"
#include "../../paper_2211_14056_b200/csrc/generated/gg_ttxg.inc"
#include "../../paper_2211_14056_b200/csrc/generated/gg_ttxgg.inc"
#include "../../paper_2211_14056_b200/csrc/generated/gg_ttxggg.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qqx_ttx.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qqx_ttxg.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qg_ttxq.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qqx_ttxgg.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qg_ttxqg.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qxg_ttxqx.inc"
#include "../../paper_2211_14056_b200/csrc/generated/qxg_ttxqxg.inc"

using namespace madme;

template <class P> struct Tables;
#define DEF_TABLES(U)                                           \
  template <> struct Tables<U> {                                \
    static const MeItem* items() { static const MeItem t[] = U##_ITEM_TABLE; return t; }        \
    static const MeMember* members() { static const MeMember t[] = U##_MEMBER_TABLE; return t; } \
    static const int* masks() { static const int t[] = U##_SUB_MASKS; return t; }       \
    static const int* kind() { static const int t[] = U##_LEG_KIND; return t; }         \
    static const int* massive() { static const int t[] = U##_LEG_MASSIVE; return t; }   \
    static const int* ext_off() { static const int t[] = U##_EXT_OFF; return t; }       \
  };
#define FOR_EACH_PROCESS(X) X(epem_mupmum) X(gg_ttx) X(gg_ttxg) X(gg_ttxgg) X(gg_ttxggg) X(qqx_ttx) X(qqx_ttxg) X(qg_ttxq) X(qqx_ttxgg) X(qg_ttxqg) X(qxg_ttxqx) X(qxg_ttxqxg)
FOR_EACH_PROCESS(DEF_TABLES)

// items [begin, end) of one stage for ONE event: the device runs them with lanes = (local variant j, event)
template <class P> void items(double* sm, int begin, int end, double mass) {
  for (int it = begin; it < end; ++it)
    for (int j = 0; j < P::VPI; ++j) {
      // all three forms of the member loop
      if (it % 3 == 1) me_run_item<1, P::VPI, P::NSLOT>(Tables<P>::items()[it], Tables<P>::members(), j, sm, mass);
      else if (it % 3 == 2) me_run_item<2, P::VPI, P::NSLOT>(Tables<P>::items()[it], Tables<P>::members(), j, sm, mass);
      else me_run_item<0, P::VPI, P::NSLOT>(Tables<P>::items()[it], Tables<P>::members(), j, sm, mass);
    }
}

// the chunked form (me_kernel.cuh::cta_me2_chunked): passes over the frozen helicities, J held whole here (the device keeps
// it in tensor memory), dots and colour called chunk by chunk exactly as the device does
template <class P> void eval_chunked(const double* mom, double* me2, long long n, double mass, double coupling, double* per_hel) {
  std::vector<double> sm(P::SMEM_DOUBLES);
  double g2 = 1;
  for (int i = 0; i < P::COUPLING_POWER; ++i) g2 *= coupling;
  const double scale = g2 / (double(P::CF_DEN) * double(P::AVG_DEN));
  constexpr int CH = P::CHUNK, NC = P::N_CHUNK;
  for (long long e = 0; e < n; ++e) {
    double s = 0;
    for (int pass = 0; pass < P::N_PASS; ++pass) {
      for (int lane = 0; lane < 32; ++lane)
        me_phase0(lane, 32, sm.data(), mom + e * 4 * P::N_EXT, P::N_EXT, P::N_SUB, Tables<P>::masks(), Tables<P>::kind(),
                  Tables<P>::massive(), Tables<P>::ext_off(), mass, P::FROZEN_MASK, P::frozen_helicities(pass));
      std::vector<double> jr(size_t(P::N_HEL_EVAL) * CH * NC, 0.0), ji(size_t(P::N_HEL_EVAL) * CH * NC, 0.0);
      int it = 0;
      for (int p = 0; p < P::N_STAGES; ++p) {
        items<P>(sm.data(), it, P::stage_end(p), mass);
        it = P::stage_end(p);
        const int r = P::stage_dots(p);
        if (r >= 0)
          for (int h = 0; h < P::N_HEL_EVAL; ++h)
            for (int c = 0; c < NC; ++c)
              if (P::has_dots(r, c)) P::dots(r, c, sm.data(), h, &jr[(size_t(h) * NC + c) * CH], &ji[(size_t(h) * NC + c) * CH]);
      }
      for (int h = 0; h < P::N_HEL_EVAL; ++h) {
        double v = 0;
        for (int ca = 0; ca < NC; ++ca) {
          const double* ar = &jr[(size_t(h) * NC + ca) * CH]; const double* ai = &ji[(size_t(h) * NC + ca) * CH];
          v += P::colour_diag(ca, ar, ai);
          for (int cb = ca + 1; cb < NC; ++cb) v += P::colour_pair(ca, cb, ar, ai, &jr[(size_t(h) * NC + cb) * CH], &ji[(size_t(h) * NC + cb) * CH]);
        }
        if (per_hel) per_hel[e * P::N_HEL + P::full_helicity(h, pass)] = v * scale;
        s += v;
      }
    }
    me2[e] = 2.0 * s * scale;
  }
}

template <class P> void eval(const double* mom, double* me2, long long n, double mass, double coupling, double* per_hel, bool split) {
  if constexpr (P::CHUNKED) {
    eval_chunked<P>(mom, me2, n, mass, coupling, per_hel);
    return;
  } else {
  std::vector<double> sm(P::SMEM_DOUBLES);
  double g2 = 1;
  for (int i = 0; i < P::COUPLING_POWER; ++i) g2 *= coupling;
  const double scale = g2 / (double(P::CF_DEN) * double(P::AVG_DEN));
  for (long long e = 0; e < n; ++e) {
    for (int lane = 0; lane < 32; ++lane)
      me_phase0(lane, 32, sm.data(), mom + e * 4 * P::N_EXT, P::N_EXT, P::N_SUB, Tables<P>::masks(), Tables<P>::kind(),
                Tables<P>::massive(), Tables<P>::ext_off(), mass);
    int it = 0;
    // both forms of the dot / colour stages: one warp per event (J whole) and two warps per event (each half of the flows)
    std::vector<double> jr(P::N_HEL_EVAL * P::N_FLOW, 0.0), ji(P::N_HEL_EVAL * P::N_FLOW, 0.0);
    constexpr int NH = P::N_FLOW_HALF;
    std::vector<double> ar(P::N_HEL_EVAL * NH, 0.0), ai(P::N_HEL_EVAL * NH, 0.0), br(P::N_HEL_EVAL * NH, 0.0), bi(P::N_HEL_EVAL * NH, 0.0);
    for (int p = 0; p < P::N_STAGES; ++p) {
      items<P>(sm.data(), it, P::stage_end(p), mass);
      it = P::stage_end(p);
      const int r = P::stage_dots(p);
      if (r >= 0)
        for (int h = 0; h < P::N_HEL_EVAL; ++h) {
          P::dots(r, sm.data(), h, &jr[h * P::N_FLOW], &ji[h * P::N_FLOW]);
          P::dots_a(r, sm.data(), h, &ar[h * NH], &ai[h * NH]);
          P::dots_b(r, sm.data(), h, &br[h * NH], &bi[h * NH]);
        }
    }
    double s = 0;
    for (int h = 0; h < P::N_HEL_EVAL; ++h) {
      double v = P::colour(&jr[h * P::N_FLOW], &ji[h * P::N_FLOW]);
      // role A: pairs inside A + A x (first chunk of B); role B: pairs inside B + (second part of B) x A in two chunks
      const double* Ar = &ar[h * NH]; const double* Ai = &ai[h * NH]; const double* Br = &br[h * NH]; const double* Bi = &bi[h * NH];
      const double va = P::colour_own_a(Ar, Ai) + P::colour_cross_a(Ar, Ai, Br, Bi);
      const double vb = P::colour_own_b(Br, Bi) + P::colour_cross_b0(Br, Bi, Ar, Ai) + P::colour_cross_b1(Br, Bi, Ar + P::CHUNK_A, Ai + P::CHUNK_A);
      if (split) v = va + vb;
      if (per_hel) per_hel[e * P::N_HEL_EVAL + h] = v * scale;
      s += v;
    }
    me2[e] = 2.0 * s * scale;
  }
  }
}

// split != 0: the two-warps-per-event form of the dot and colour stages (each warp half of the colour flows)
extern "C" int host_me_eval(const char* proc, const double* mom, double* me2, long long n, double mass, double coupling,
                            double* per_hel, int split) {
#define TRY(P) if (!strcmp(proc, #P)) { eval<P>(mom, me2, n, mass, coupling, per_hel, split != 0); return 0; }
  FOR_EACH_PROCESS(TRY)
#undef TRY
  return -1;
}
