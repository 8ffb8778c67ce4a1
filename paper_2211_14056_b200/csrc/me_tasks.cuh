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
//                    ITS OWN legs ("helicity recycling").  Storage is in GROUPS of 4 lines x 128 B, one line per
//                    component; o owns nv consecutive 16-byte slots of each line:
//                    component c, variant v  ->  double offset  OFF_o + 16 c + 2 v        (ME_WF_STRIDE = 16)
//                    so that the 32 lanes' 16-byte loads of one component fall into <= 128 contiguous bytes (one
//                    shared-memory wavefront) and the four components are one address + immediate offsets.
//   Leg 0 is fixed at helicity +1 (parity: |M(-h)|^2 = |M(h)|^2, the sum is doubled at the end), so
//   variant index v = sum_k b_{l_k} 2^k over the legs l_0 < l_1 < ... of S OTHER THAN LEG 0, b = 0 for helicity -1,
//   1 for +1, and nv = 2^(number of those legs).
//   The first BASE_DOUBLES hold what every round reads (subset blocks, external wavefunctions, the currents that feed
//   other currents); the rest is the ROUND region, reused by successive rounds of leg splits (gen/emit.py).
//
// The steps:
//   a5  me_phase0      : K_S and propagator denominators for every subset, external wavefunctions
//   a6  me_run_row     : off-shell currents and their combinations, one (object, variant) task per thread, stage by stage
//   a7-a10             : generated straight-line code (csrc/generated/*.inc: dots, colour), one helicity per lane
#pragma once
#include "helas.cuh"

namespace madme {

// One task = one (object, helicity variant), encoded in 128 bits so that a lane fetches its task with one load:
//   x: out | a << 16                      (offsets in doubles into the event's scratch)
//   y: b   | c << 16
//   z: ksub_out | ksub_a << 8 | ksub_b << 16 | op << 24 | massive << 27 | open << 28      (ksub = subset index)
//   w: n_members << 16 | phase codes (2 bits each) << 20                                    (OP_COMBO)
// OP_VVVV writes the three colour terms of a four-gluon current: out, (z >> 8) & 0xffff and w & 0xffff.
// OP_COMBO: out = sum_j i^{k_j} member_j with members (a, b, c, and a fourth in z & 0xffff).  Rows come in groups of
// one op (padded with OP_NOP to multiples of 4 rows), groups in stages; a barrier separates stages.
struct MeRow { unsigned x, y, z, w; };
enum MeOp { OP_FFV_ROW = 0, OP_FFV_COL = 1, OP_FFV_VEC = 2, OP_VVV = 3, OP_VVVV = 4, OP_COMBO = 5, OP_NOP = 7 };

constexpr int ME_WF_STRIDE = 16;  // doubles between the components of a stored wavefunction (one 128-byte line)
ME_HD wf4 ld_wf(const double* p) {
  constexpr int stride = ME_WF_STRIDE;
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
ME_HD void st_wf(double* p, const wf4& w) {
  constexpr int stride = ME_WF_STRIDE;
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
// Work items idx, idx + step, ... (subsets, then legs) of ONE event.
ME_HD void me_phase0(int idx, int step, double* sm, const double* mom, int n_ext, int n_sub, const int* sub_masks,
                     const int* leg_kind, const int* leg_massive, const int* ext_off, double mass) {
  for (int s = idx; s < n_sub; s += step) {
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
  for (int l = idx; l < n_ext; l += step) {
    wf4 w[2];
    external_wavefunction(leg_kind[l], mom + 4 * l, leg_massive[l] ? mass : 0.0, w);
    if (l == 0) {
      st_wf(sm + ext_off[0], w[1]);  // leg 0: helicity +1 only (parity)
    } else {
      st_wf(sm + ext_off[l], w[0]);
      st_wf(sm + ext_off[l] + 2, w[1]);
    }
  }
}

// i^k x
ME_HD cplx times_ik(cplx x, int k) {
  const double re = (k & 1) ? -x.im : x.re, im = (k & 1) ? x.re : x.im;
  return mk((k & 2) ? -re : re, (k & 2) ? -im : im);
}

// acc += i^k x for a stored wavefunction: i^k = cr + i ci with cr, ci in {0, +-1} assembled from the bits of k (no
// int->double conversion, no select cascade), then four FMAs per component
ME_HD void combo_add(wf4& acc, const double* p, int k) {
  const wf4 x = ld_wf(p);
#if defined(__CUDA_ARCH__)
  const int one = 0x3FF00000 | ((k & 2) << 30);  // high word of +1.0 (k = 0, 1) or -1.0 (k = 2, 3)
  const double cr = __hiloint2double((k & 1) ? 0 : one, 0), ci = __hiloint2double((k & 1) ? one : 0, 0);
#else
  const double sgn = (k & 2) ? -1.0 : 1.0, cr = (k & 1) ? 0.0 : sgn, ci = (k & 1) ? sgn : 0.0;
#endif
  for (int c = 0; c < 4; ++c) {
    acc.c[c].re = fma(cr, x.c[c].re, fma(-ci, x.c[c].im, acc.c[c].re));
    acc.c[c].im = fma(cr, x.c[c].im, fma(ci, x.c[c].re, acc.c[c].im));
  }
}

// a6: one task
ME_HD void me_run_row(const MeRow r, double* sm, double mass) {
  const int op = (r.z >> 24) & 7;
  if (op == OP_NOP) return;
  const int out = r.x & 0xffff;
  const wf4 A = ld_wf(sm + (r.x >> 16));
  if (op == OP_COMBO) {
    // colour-ordered combination of currents over the same legs (same variant); members 2 and 3 are optional
    const int n = (r.w >> 16) & 15;
    wf4 acc = A;  // the first member always enters with coefficient 1
    combo_add(acc, sm + (r.y & 0xffff), (r.w >> 22) & 3);
    if (n > 2) combo_add(acc, sm + (r.y >> 16), (r.w >> 24) & 3);
    if (n > 3) combo_add(acc, sm + (r.z & 0xffff), (r.w >> 26) & 3);
    st_wf(sm + out, acc);
    return;
  }
  const wf4 B = ld_wf(sm + (r.y & 0xffff));
  const double* ks = sm + 8 * (r.z & 0xff);
  const bool massive = (r.z >> 27) & 1;
  const bool open = (r.z >> 28) & 1;  // the current stops at its vertex: no propagator (U side of a propagator cut)
  const double m = massive ? mass : 0.0;
  const double invk2 = open ? 1.0 : ks[4];
  // open and propagated rows sit in different groups (gen/emit.py), so these branches are warp-uniform
  if (op == OP_FFV_ROW) {
    const wf4 x = slash_row(A, B);
    if (open) st_wf(sm + out, x);
    else st_wf(sm + out, prop_row(ld_k(ks), -1.0, m, massive ? ks[5] : ks[4], x));
  } else if (op == OP_FFV_COL) {
    const wf4 x = slash_col(B, A);
    if (open) st_wf(sm + out, x);
    else st_wf(sm + out, prop_col(ld_k(ks), 1.0, m, massive ? ks[5] : ks[4], x));
  } else if (op == OP_FFV_VEC) {
    st_wf(sm + out, ffv_vec(A, B, invk2));
  } else if (op == OP_VVV) {
    st_wf(sm + out, vvv_vec(A, ld_k(sm + 8 * ((r.z >> 8) & 0xff)), B, ld_k(sm + 8 * ((r.z >> 16) & 0xff)), invk2));
  } else {
    const wf4 C = ld_wf(sm + (r.y >> 16));
    wf4 t1, t2, t3;
    vvvv_vec(A, B, C, invk2, t1, t2, t3);
    st_wf(sm + out, t1);
    st_wf(sm + ((r.z >> 8) & 0xffff), t2);
    st_wf(sm + (r.w & 0xffff), t3);
  }
}

// rows [begin, end) of one stage, 32 lanes at a time (host emulation and reference semantics of the device loop)
ME_HD void me_run_rows(int lane, double* sm, const MeRow* tab, int begin, int end, double mass) {
  for (int i = begin + lane; i < end; i += 32) me_run_row(tab[i], sm, mass);
}

}  // namespace madme
