// me_tasks.cuh — per-event scratch layout and the table-driven cooperative steps of me_eval.
//
// One warp owns one event ("parallelized in the event axis"; the 32 lanes of the warp are
// 32 helicity combinations of that event — SURVEY.md §7 "hard parts", option B).  The event's
// wavefunctions live in a private slice of SHARED MEMORY and never touch HBM: that is the paper's
// memory-footprint point taken to its limit.
//
// Scratch layout of one event (doubles), produced by gen/emit.py for each process:
//   subset blocks  : 8 doubles per used leg subset S:  K_S[4], 1/K_S^2, 1/(K_S^2 - m_t^2), pad, pad
//   wavefunctions  : object o over the leg set S has one helicity variant per combination of the helicities of
//                    ITS OWN legs ("helicity recycling"), stored as
//                    [component c = 0..3][variant v][re, im]   ->  double offset  OFF_o + 2*(c*nv + v)
//                    so that the 32 lanes' 16-byte loads of one component fall into <= 128 contiguous bytes.
//   Leg 0 is fixed at helicity +1 (parity: |M(-h)|^2 = |M(h)|^2, the sum is doubled at the end), so
//   variant index v = sum_k b_{l_k} 2^k over the legs l_0 < l_1 < ... of S OTHER THAN LEG 0, b = 0 for helicity -1,
//   1 for +1, and nv = 2^(number of those legs).
//   The first PERSISTENT_DOUBLES hold what the closings read; the rest is a transient region that the top-level
//   currents of successive rounds reuse once their colour-ordered combinations have been formed.
//
// The steps:
//   a5  me_phase0      : K_S and propagator denominators for every subset, external wavefunctions
//   a6  P::stage(s)    : off-shell currents and their combinations, one (object, variant) task per lane, stage by stage
//   a7-a10             : generated straight-line code (csrc/generated/*.inc), one helicity per lane
#pragma once
#include "helas.cuh"

namespace madme {

constexpr int ME_TASK_INTS = 16;
// task row: 0 out, 1 out_stride, 2 a, 3 a_stride, 4 b, 5 b_stride, 6 c, 7 c_stride,
//           8 ksub_out, 9 ksub_a, 10 ksub_b, 11 massive, 12 out2, 13 out3, 14 ksub_c, 15 unpropagated
// combo row: 0 out, 1 stride, 2 n, then n x (input offset, k) : out = sum_j i^k_j in_j
#if defined(__CUDA_ARCH__)
#define ME_FENCE() asm volatile("" ::: "memory")  // keeps ptxas from hoisting every shared-memory load to the top
#else
#define ME_FENCE()
#endif
enum MeOp { OP_FFV_ROW = 0, OP_FFV_COL = 1, OP_FFV_VEC = 2, OP_VVV = 3, OP_VVVV = 4 };

ME_HD wf4 ld_wf(const double* p, int stride) {
  wf4 w;
#if defined(__CUDA_ARCH__)
  for (int c = 0; c < 4; ++c) {
    const double2 z = *reinterpret_cast<const double2*>(p + c * stride);
    w.c[c].re = z.x; w.c[c].im = z.y;
  }
#else
  for (int c = 0; c < 4; ++c) { w.c[c].re = p[c * stride]; w.c[c].im = p[c * stride + 1]; }
#endif
  return w;
}
ME_HD void st_wf(double* p, int stride, const wf4& w) {
#if defined(__CUDA_ARCH__)
  for (int c = 0; c < 4; ++c) *reinterpret_cast<double2*>(p + c * stride) = make_double2(w.c[c].re, w.c[c].im);
#else
  for (int c = 0; c < 4; ++c) { p[c * stride] = w.c[c].re; p[c * stride + 1] = w.c[c].im; }
#endif
}
ME_HD vec4 ld_k(const double* p) {
  vec4 k;
#if defined(__CUDA_ARCH__)
  const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
  k.v[0] = a.x; k.v[1] = a.y; k.v[2] = b.x; k.v[3] = b.y;
#else
  for (int i = 0; i < 4; ++i) k.v[i] = p[i];
#endif
  return k;
}

// a5: subset momenta + denominators, external wavefunctions.  `mom` = this event's [n_ext][4] (E,px,py,pz),
// physical momenta; legs 0,1 incoming.  sub_masks[s] = bitmask of legs of subset s (block s at sm + 8 s).
ME_HD void me_phase0(int lane, double* sm, const double* mom, int n_ext, int n_sub, const int* sub_masks,
                     const int* leg_kind, const int* leg_massive, const int* ext_off, double mass) {
  for (int s = lane; s < n_sub; s += 32) {
    const int m = sub_masks[s];
    double K[4] = {0.0, 0.0, 0.0, 0.0};
    int cnt = 0;
    for (int l = 0; l < n_ext; ++l)
      if ((m >> l) & 1) {
        const double sg = (l < 2) ? 1.0 : -1.0;  // all-incoming convention
        for (int i = 0; i < 4; ++i) K[i] = fma(sg, mom[4 * l + i], K[i]);
        ++cnt;
      }
    double* o = sm + 8 * s;
    for (int i = 0; i < 4; ++i) o[i] = K[i];
    if (cnt > 1) {
      const double k2 = fma(K[0], K[0], -fma(K[1], K[1], fma(K[2], K[2], K[3] * K[3])));
      o[4] = 1.0 / k2;
      o[5] = 1.0 / fma(-mass, mass, k2);
    } else {
      o[4] = 0.0; o[5] = 0.0;
    }
  }
  for (int l = lane; l < n_ext; l += 32) {
    wf4 w[2];
    external_wavefunction(leg_kind[l], mom + 4 * l, leg_massive[l] ? mass : 0.0, w);
    if (l == 0) {
      st_wf(sm + ext_off[0], 2, w[1]);  // leg 0: helicity +1 only (parity)
    } else {
      st_wf(sm + ext_off[l], 4, w[0]);
      st_wf(sm + ext_off[l] + 2, 4, w[1]);
    }
  }
}

// a6: one off-shell current variant
ME_HD void me_run_task(int op, double* sm, const int* t, double mass) {
  const wf4 A = ld_wf(sm + t[2], t[3]);
  const wf4 B = ld_wf(sm + t[4], t[5]);
  const double* ks = sm + t[8];
  const double m = t[11] ? mass : 0.0;
  const bool open = t[15] != 0;  // the current stops at its vertex: no propagator (the U side of a propagator cut)
  const double invk2 = open ? 1.0 : ks[4];
  if (op == OP_FFV_ROW) {
    const wf4 x = slash_row(A, B);
    st_wf(sm + t[0], t[1], open ? x : prop_row(ld_k(ks), -1.0, m, t[11] ? ks[5] : ks[4], x));
  } else if (op == OP_FFV_COL) {
    const wf4 x = slash_col(B, A);
    st_wf(sm + t[0], t[1], open ? x : prop_col(ld_k(ks), 1.0, m, t[11] ? ks[5] : ks[4], x));
  } else if (op == OP_FFV_VEC) {
    st_wf(sm + t[0], t[1], ffv_vec(A, B, invk2));
  } else if (op == OP_VVV) {
    st_wf(sm + t[0], t[1], vvv_vec(A, ld_k(sm + t[9]), B, ld_k(sm + t[10]), invk2));
  } else {
    const wf4 C = ld_wf(sm + t[6], t[7]);
    wf4 t1, t2, t3;
    vvvv_vec(A, B, C, invk2, t1, t2, t3);
    st_wf(sm + t[0], t[1], t1);
    st_wf(sm + t[12], t[1], t2);
    st_wf(sm + t[13], t[1], t3);
  }
}

// all tasks [begin, end) of one (level, op) group, 32 lanes at a time
ME_HD void me_run_group(int op, int lane, double* sm, const int* tab, int begin, int end, double mass) {
  for (int i = begin + lane; i < end; i += 32) me_run_task(op, sm, tab + ME_TASK_INTS * i, mass);
}

// colour-ordered combinations: out = sum_j i^{k_j} in_j (same leg set, same variant)
ME_HD void me_run_combos(int lane, double* sm, const int* ctab, int begin, int end) {
  for (int i = begin + lane; i < end; i += 32) {
    const int* t = ctab + ME_TASK_INTS * i;
    wf4 acc = ld_wf(sm + t[3], t[1]);  // first member always enters with coefficient 1
    for (int j = 1; j < t[2]; ++j) {
      const wf4 x = ld_wf(sm + t[3 + 2 * j], t[1]);
      const int k = t[4 + 2 * j];
      for (int c = 0; c < 4; ++c) {
        const double re = (k & 1) ? -x.c[c].im : x.c[c].re, im = (k & 1) ? x.c[c].re : x.c[c].im;
        acc.c[c].re += (k & 2) ? -re : re;
        acc.c[c].im += (k & 2) ? -im : im;
      }
    }
    st_wf(sm + t[0], t[1], acc);
  }
}

}  // namespace madme
