// me_tasks.cuh — per-event scratch layout and the table-driven cooperative steps of me_eval.
//
// A CTA works on W events at a time ("parallelized in the event axis").  An event's wavefunctions live in
// a private slice of SHARED MEMORY and never touch HBM: that is the paper's memory-footprint point (PAPER.md:9,
// 62-64) taken to its limit.
//
// Scratch layout of one event (doubles), produced by gen/emit.py for each process:
//   subset blocks  : 8 doubles per used leg subset S:  K_S[4], the propagator denominator 1/(K_S^2 - m^2) of the currents
//                    over S (m = m_t on the massive quark line, else 0; only where a propagated current exists), pads
//   wavefunctions  : object o over the leg set S has one helicity variant per combination of the helicities of
//                    ITS OWN legs ("helicity recycling").  Storage is in GROUPS of 4 lines x 128 B, one line per
//                    component; o owns nv consecutive 16-byte slots of each line:
//                    component c, variant v  ->  double offset  OFF_o + 16 c + 2 v        (ME_WF_STRIDE = 16)
//                    so that the 32 lanes' 16-byte loads of one component fall into <= 128 contiguous bytes (one
//                    shared-memory wavefront) and the four components are one address + immediate offsets.
//   Leg 0 is fixed at helicity +1 (parity: |M(-h)|^2 = |M(h)|^2, the sum is doubled at the end), so
//   variant index v = sum_k b_{l_k} 2^k over the legs l_0 < l_1 < ... of S OTHER THAN LEG 0, b = 0 for helicity -1,
//   1 for +1, and nv = 2^(number of those legs).
//   Only what somebody reads is stored: the first BASE_DOUBLES hold what every round reads (subset blocks, external
//   wavefunctions, the currents that feed other currents); the rest is the ROUND region, reused by successive rounds
//   of leg splits, and holds the operands of the round's propagator-cut dot products (gen/emit.py).
//
// The steps:
//   a5  me_phase0      : K_S and propagator denominators for every subset, external wavefunctions
//   a6  me_run_item    : one ITEM = up to 4 colour-ordered currents over one leg set, for one helicity variant per
//                        lane: the bare vertices of the Feynman subdiagrams that enter them are evaluated in registers
//                        and summed with their {+-1, +-i} coefficients, the common propagator is applied once per sum
//   a7-a10             : generated straight-line code (csrc/generated/*.inc: dots, colour), one helicity per lane
#pragma once
#include "helas.cuh"

namespace madme {

// One item (16 B), warp-uniform:
//   w0: n_members | n_out << 8 | kind << 12 | massive << 15 | nv << 16 | vbase << 24
//   w1: first_member | ksub_out << 16                      (ksub = subset index: block at sm + 8 ksub)
//   w2: out0 | out1 << 16,  w3: out2 | out3 << 16          (offsets in doubles into the event's scratch, variant 0)
// One member (32 B) = one bare vertex:
//   w0: op | ksub_a << 8 | ksub_b << 16
//   w1: a | b << 16,   w2: c,   w3: vmap_a,   w5: vmap_b,   w6: vmap_c
//        (vmap: which variant of the argument enters local variant j of the outputs.  VPI = 4: one byte per j, the
//        variant's offset in 16-byte slots; VPI = 8: four bits per j, the variant index)
//   w4: code of term 0 | code of term 1 << 9 | code of term 2 << 18      (see acc_term; terms 1, 2 exist for the
//        four-gluon vertex only)
struct MeItem { unsigned w0, w1, w2, w3; };
struct MeMember { unsigned w[8]; };
enum MeOp { OP_SLASH_ROW = 0, OP_SLASH_COL = 1, OP_FFV_VEC = 2, OP_VVV = 3, OP_VVVV = 4 };
enum MeKind { KIND_VEC = 0, KIND_ROW = 1, KIND_COL = 2, KIND_OPEN = 3 };
constexpr int ME_NSLOT = 4;   // most accumulators of an item (gen/emit.py::NSLOT; a process may be generated with 2)

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
// physical momenta; legs 0,1 incoming.  sub_masks[s] = bitmask of legs of subset s (block s at sm + 8 s) | flags << 16:
// flag 1 = some propagated current lives on S (the denominator is needed), flag 2 = that line is massive.
// Work items idx, idx + step, ... (subsets, then legs) of ONE event.
// frozen_mask: legs whose helicity is fixed (leg 0 by parity; more for processes evaluated in passes); their fixed
// helicities are the bits of frozen_hel at the leg positions, and only that wavefunction is stored.
ME_HD void me_phase0(int idx, int step, double* sm, const double* mom, int n_ext, int n_sub, const int* sub_masks,
                     const int* leg_kind, const int* leg_massive, const int* ext_off, double mass,
                     unsigned frozen_mask = 1u, unsigned frozen_hel = 1u) {
  // rolled: this runs once per event and must not crowd the instruction cache of the item and dot stages
#if defined(__CUDA_ARCH__)
#pragma unroll 1
#endif
  for (int s = idx; s < n_sub; s += step) {
    const int m = sub_masks[s];
    double K[4] = {0.0, 0.0, 0.0, 0.0};
    for (int l = 0; l < n_ext; ++l)
      if ((m >> l) & 1) {
        const double sg = (l < 2) ? 1.0 : -1.0;  // all-incoming convention
        for (int i = 0; i < 4; ++i) K[i] = fma(sg, mom[4 * l + i], K[i]);
      }
    double* o = sm + 8 * s;
    for (int i = 0; i < 4; ++i) o[i] = K[i];
    if ((m >> 16) & 1) {
      const double k2 = fma(K[0], K[0], -fma(K[1], K[1], fma(K[2], K[2], K[3] * K[3])));
      o[4] = 1.0 / (((m >> 17) & 1) ? fma(-mass, mass, k2) : k2);
    }
  }
#if defined(__CUDA_ARCH__)
#pragma unroll 1
#endif
  for (int l = idx; l < n_ext; l += step) {
    wf4 w[2];
    external_wavefunction(leg_kind[l], mom + 4 * l, leg_massive[l] ? mass : 0.0, w);
    if ((frozen_mask >> l) & 1u) {
      st_wf(sm + ext_off[l], w[(frozen_hel >> l) & 1u]);  // one helicity only (leg 0: +1, parity)
    } else {
      st_wf(sm + ext_off[l], w[0]);
      st_wf(sm + ext_off[l] + 2, w[1]);
    }
  }
}

// A term x of a bare vertex enters the item's accumulators as  acc_s += e_s (i^b x),  e_s in {0, +1, -1}: its 9-bit code
// is  b | sign_0 << 1 | sign_1 << 3 | sign_2 << 5 | sign_3 << 7  with sign 0 none, 1 plus, 2 minus (gen/emit.py:
// Task.solve_phases).  Everything here is warp-uniform; the only branches are on b and on "more than two currents".
ME_HD double sign_of(unsigned code2) {   // 0 -> 0.0, 1 -> +1.0, 2 -> -1.0
#if defined(__CUDA_ARCH__)
  return __hiloint2double(static_cast<int>((code2 ? 0x3FF00000u : 0u) | ((code2 & 2u) << 30)), 0);
#else
  return code2 == 0 ? 0.0 : (code2 == 1 ? 1.0 : -1.0);
#endif
}
ME_HD void acc_plain(wf4& acc, const wf4& x, double e) {
  for (int c = 0; c < 4; ++c) { acc.c[c].re = fma(e, x.c[c].re, acc.c[c].re); acc.c[c].im = fma(e, x.c[c].im, acc.c[c].im); }
}
ME_HD void acc_times_i(wf4& acc, const wf4& x, double e) {
  for (int c = 0; c < 4; ++c) { acc.c[c].re = fma(-e, x.c[c].im, acc.c[c].re); acc.c[c].im = fma(e, x.c[c].re, acc.c[c].im); }
}
template <int NS> ME_HD void acc_term(wf4 (&acc)[NS], const wf4& x, unsigned code, bool wide) {
  const double e0 = sign_of((code >> 1) & 3u), e1 = sign_of((code >> 3) & 3u);
  if (code & 1u) {
    acc_times_i(acc[0], x, e0);
    acc_times_i(acc[1], x, e1);
    if (NS > 2 && wide) {
      acc_times_i(acc[NS > 2 ? 2 : 0], x, sign_of((code >> 5) & 3u));
      acc_times_i(acc[NS > 2 ? 3 : 0], x, sign_of((code >> 7) & 3u));
    }
  } else {
    acc_plain(acc[0], x, e0);
    acc_plain(acc[1], x, e1);
    if (NS > 2 && wide) {
      acc_plain(acc[NS > 2 ? 2 : 0], x, sign_of((code >> 5) & 3u));
      acc_plain(acc[NS > 2 ? 3 : 0], x, sign_of((code >> 7) & 3u));
    }
  }
}

// a6: one item for local variant j (0 .. VPI-1) of one event (scratch at sm).  PREFETCH: fetch the operands of member
// i + 1 before member i is evaluated (32 more registers; for CTAs with two warps per scheduler).
// double offset of helicity variant v inside a stored object (gen/emit.py::voff): 16-byte slots of a 128-byte line; an
// object with 16 variants continues in the next group of four lines
ME_HD int me_voff(unsigned v) { return static_cast<int>(2u * (v & 7u) + 64u * (v >> 3)); }
// double offset of the variant of an argument that enters local variant j of the item (tables above)
template <int VPI> ME_HD int me_arg_off(unsigned word, int j) {
  return VPI == 4 ? static_cast<int>(2u * ((word >> (8 * j)) & 0xffu)) : me_voff((word >> (4 * j)) & 15u);
}
template <int PREFETCH, int VPI = 4, int NS = ME_NSLOT>
ME_HD void me_run_item(const MeItem H, const MeMember* __restrict__ members, int j, double* __restrict__ sm, double mass) {
#define ME_LD_ARG(off) ld_wf(sm + (off))
  const int n_mem = H.w0 & 0xff;
  const int nv = (H.w0 >> 16) & 0xff, v = static_cast<int>(H.w0 >> 24) + j;
  if (n_mem == 0 || v >= nv) return;
  const int n_out = (H.w0 >> 8) & 0xf, kind = (H.w0 >> 12) & 7;
  const bool wide = n_out > 2;
  wf4 acc[NS];
  for (int s = 0; s < NS; ++s)
    for (int c = 0; c < 4; ++c) acc[s].c[c] = mk(0.0, 0.0);
  const MeMember* m = members + (H.w1 & 0xffff);
  unsigned w0 = m->w[0], w2 = m->w[2], w4 = m->w[4], w6 = m->w[6];
  wf4 A, B;
  {
    const unsigned w1 = m->w[1];
    A = ME_LD_ARG((w1 & 0xffff) + me_arg_off<VPI>(m->w[3], j));
    B = ME_LD_ARG((w1 >> 16) + me_arg_off<VPI>(m->w[5], j));
  }
#if defined(__CUDA_ARCH__)
#pragma unroll 1
#endif
  for (int i = 0; i < n_mem; ++i) {
    const unsigned c0 = w0, c2 = w2, c4 = w4, c6 = w6;
    const wf4 a = A, b = B;
    // the operands of member i + 1: PREFETCH 1 before member i is evaluated (copies), 2 between its vertex and its
    // accumulation (no copies: a and b are dead by then), 0 after it
#define ME_FETCH_NEXT()                                                                         \
    if (i + 1 < n_mem) {                                                                        \
      ++m;                                                                                      \
      const unsigned w1 = m->w[1];                                                              \
      w0 = m->w[0]; w2 = m->w[2]; w4 = m->w[4]; w6 = m->w[6];                                    \
      A = ME_LD_ARG((w1 & 0xffff) + me_arg_off<VPI>(m->w[3], j));                                \
      B = ME_LD_ARG((w1 >> 16) + me_arg_off<VPI>(m->w[5], j));                                   \
    }
    if (PREFETCH == 1) { ME_FETCH_NEXT() }
    const int op = c0 & 0xff;
    if (PREFETCH == 2) {
      wf4 t1, t2, t3;
      if (op == OP_SLASH_ROW) t1 = slash_row(a, b);
      else if (op == OP_SLASH_COL) t1 = slash_col(b, a);
      else if (op == OP_FFV_VEC) t1 = ffv_vec_bare(a, b);
      else if (op == OP_VVV) t1 = vvv_vec_bare(a, ld_k(sm + 8 * ((c0 >> 8) & 0xff)), b, ld_k(sm + 8 * ((c0 >> 16) & 0xff)));
      else {
        const wf4 C = ME_LD_ARG((c2 & 0xffff) + me_arg_off<VPI>(c6, j));
        vvvv_vec_bare(a, b, C, t1, t2, t3);
      }
      ME_FETCH_NEXT()
      acc_term(acc, t1, c4 & 0x1ffu, wide);
      if (op == OP_VVVV) {
        acc_term(acc, t2, (c4 >> 9) & 0x1ffu, wide);
        acc_term(acc, t3, (c4 >> 18) & 0x1ffu, wide);
      }
    } else {
    if (op == OP_SLASH_ROW) {
      acc_term(acc, slash_row(a, b), c4 & 0x1ffu, wide);
    } else if (op == OP_SLASH_COL) {
      acc_term(acc, slash_col(b, a), c4 & 0x1ffu, wide);
    } else if (op == OP_FFV_VEC) {
      acc_term(acc, ffv_vec_bare(a, b), c4 & 0x1ffu, wide);
    } else if (op == OP_VVV) {
      acc_term(acc, vvv_vec_bare(a, ld_k(sm + 8 * ((c0 >> 8) & 0xff)), b, ld_k(sm + 8 * ((c0 >> 16) & 0xff))), c4 & 0x1ffu, wide);
    } else {
      const wf4 C = ME_LD_ARG((c2 & 0xffff) + me_arg_off<VPI>(c6, j));
      wf4 t1, t2, t3;
      vvvv_vec_bare(a, b, C, t1, t2, t3);
      acc_term(acc, t1, c4 & 0x1ffu, wide);
      acc_term(acc, t2, (c4 >> 9) & 0x1ffu, wide);
      acc_term(acc, t3, (c4 >> 18) & 0x1ffu, wide);
    }
    }
    if (PREFETCH == 0) { ME_FETCH_NEXT() }
#undef ME_FETCH_NEXT
#undef ME_LD_ARG
  }
  // the common propagator, once per colour-ordered current
  const double* ks = sm + 8 * (H.w1 >> 16);
  const unsigned outs[4] = {H.w2 & 0xffff, H.w2 >> 16, H.w3 & 0xffff, H.w3 >> 16};
  if (kind == KIND_OPEN) {
    for (int s = 0; s < NS; ++s)
      if (s < n_out) st_wf(sm + outs[s] + me_voff(v), acc[s]);
  } else if (kind == KIND_VEC) {
    const double f = ks[4];
    for (int s = 0; s < NS; ++s)
      if (s < n_out) {
        wf4 y;
        for (int c = 0; c < 4; ++c) y.c[c] = f * acc[s].c[c];
        st_wf(sm + outs[s] + me_voff(v), y);
      }
  } else {
    const bool massive = (H.w0 >> 15) & 1;
    const double mm = massive ? mass : 0.0, f = ks[4];
    const vec4 K = ld_k(ks);
    if (kind == KIND_ROW) {
      for (int s = 0; s < NS; ++s)
        if (s < n_out) st_wf(sm + outs[s] + me_voff(v), prop_row(K, -1.0, mm, f, acc[s]));
    } else {
      for (int s = 0; s < NS; ++s)
        if (s < n_out) st_wf(sm + outs[s] + me_voff(v), prop_col(K, 1.0, mm, f, acc[s]));
    }
  }
}

}  // namespace madme
