// me_kernel.cuh — the me_eval kernel: a CTA of W = 8 warps evaluates 8 events at a time.
//
// the tensorised generator materialises every wavefunction as an HBM tensor over events and
// its footprint grows with the number of diagrams; the paper's CUDA op keeps them in per-thread storage
// (PAPER.md:70-72).  Here an event's wavefunctions live in a private slice of SHARED MEMORY (BASE + one ROUND
// region, generated/*.inc), every off-shell current is computed once per combination of the helicities of ITS OWN
// legs ("helicity recycling", me_tasks.cuh) and HBM sees 32 n_ext bytes in and 8 bytes out per event.
//
// Two mappings alternate inside the CTA (a __syncthreads between them):
//   current stages (a5, a6): warp w runs items w, w + W, ... of the stage; the 32 lanes of an item are 4 helicity
//       variants x 8 events, so the item (its vertices, operands, coefficients) is warp-uniform: no divergence, no
//       per-lane task decoding;
//   dot stages (a7-a10): warp w owns event w, lane = helicity combination, J (the colour-flow vector) in registers.
// Between the dot stages of successive rounds J is PARKED IN TENSOR MEMORY (tcgen05.st / tcgen05.ld, 4 N_FLOW 32-bit
// columns per warp), so that the current stages have the whole register file for their accumulators.
//
// Compiled once per process: the including translation unit defines MADME_PROC (build.py).
#pragma once
#ifndef MADME_PROC
#error "compile with -DMADME_PROC=<process>"
#endif
#define MADME_STR_(x) #x
#define MADME_STR(x) MADME_STR_(x)
#define MADME_INC(p) MADME_STR(generated/p.inc)
#include MADME_INC(MADME_PROC)
#include "tmem.cuh"
#ifndef MADME_PREFETCH_CHUNKED
#define MADME_PREFETCH_CHUNKED 1   // g g -> t tbar g g g: 1.45 M events/s (0: 1.39 M)
#endif
#ifndef MADME_PREFETCH
#define MADME_PREFETCH 0   // 0: the next member's operands are fetched after the accumulation (58.7 M events/s); 1: one member ahead, copied (56.9 M); 2: between vertex and accumulation (56.8 M)
#endif

#ifndef MADME_PREFETCH_MOMENTA
#define MADME_PREFETCH_MOMENTA 1   // me_eval: the next batch's momenta are fetched (cp.async) while this batch is computed
#endif
#ifndef MADME_STRIDE8
#define MADME_STRIDE8 8   // doubles mod 16 between the events of a four-event CTA
#endif

namespace madme {

#define MADME_CAT2_(a, b) a##b
#define MADME_CAT2(a, b) MADME_CAT2_(a, b)
#define MADME_TAB(suffix) MADME_CAT2(MADME_PROC, suffix)   // the table macros of generated/<process>.inc: <process>_ITEM_TABLE, ...

// the process's tables: items and members in constant memory (every lane of a warp reads the same entry), the rest
// in global memory (read once per event by phase 0)
__constant__ MeItem c_items[] = MADME_TAB(_ITEM_TABLE);
__constant__ MeMember c_members[] = MADME_TAB(_MEMBER_TABLE);
__device__ const int d_masks[] = MADME_TAB(_SUB_MASKS);
__device__ const int d_kind[] = MADME_TAB(_LEG_KIND);
__device__ const int d_massive[] = MADME_TAB(_LEG_MASSIVE);
__device__ const int d_extoff[] = MADME_TAB(_EXT_OFF);

// doubles of shared memory per event: momenta [n_ext][4] + the generated scratch layout; the stride between the
// events of a CTA is = 2 doubles (16 B) mod 16 doubles (128 B), so that the same object of neighbouring events
// (neighbouring lanes in the current stages) falls into different banks.
template <class P> struct EventSmem {
  static constexpr int RAW = 4 * P::N_EXT + P::SMEM_DOUBLES;
  // eight events: 16 B mod 128 B; four events (eight variants = one line per event and component): half a line
  static constexpr int DOUBLES = ((RAW + 13) / 16) * 16 + (P::VPI == 8 ? MADME_STRIDE8 : 2);
};

// Events per CTA: P::W_EVENTS (gen/emit.py: the item tables are laid out for it; 8, or 4 for g g -> t tbar g g g).  A CTA
// has P::N_WARPS >= W_EVENTS warps: all of them run items, the first W_EVENTS own one event each in the dot stages.

// J in tensor memory: warp w owns TMEM lanes 32 (w % 4) .. +31 and the column block w / 4 (REGS columns: 4 per colour
// flow it holds).  With P::SPLIT_J an event has TWO warps (w and w + 8, same lanes, neighbouring blocks), each holding
// the flows of one half; the halves meet once, for J^dagger CF J, by reading the partner's block.
template <class P> struct JPark {
  static constexpr int NFW = P::SPLIT_J ? P::N_FLOW_HALF : P::N_FLOW;   // flows per warp
  static constexpr bool ON = P::N_ROUNDS > 1 || P::SPLIT_J || P::CHUNKED;
  static constexpr int REGS = 4 * NFW;                             // 32-bit columns per warp
  // allocation: a power of two >= 32; chunked form: one column block per event of a sub-partition
  static constexpr int COLS = tmem_cols(P::CHUNKED ? ((P::W_EVENTS + 3) / 4) * 4 * P::CHUNK * P::N_CHUNK : (P::N_WARPS / 4) * REGS);
  static __device__ __forceinline__ uint32_t addr(uint32_t base, int warp) {
    return base + (static_cast<uint32_t>(32 * (warp & 3)) << 16) + (warp >> 2) * REGS;
  }
  static __device__ __forceinline__ void park(uint32_t base, int warp, const double* jr, const double* ji) {
    uint32_t r[REGS];
#pragma unroll
    for (int f = 0; f < NFW; ++f) {
      r[4 * f] = __double2loint(jr[f]); r[4 * f + 1] = __double2hiint(jr[f]);
      r[4 * f + 2] = __double2loint(ji[f]); r[4 * f + 3] = __double2hiint(ji[f]);
    }
    tmem_store<REGS>(addr(base, warp), r);
  }
  // N flows starting at flow `first` of the block of warp `owner`
  template <int N> static __device__ __forceinline__ void load(uint32_t base, int owner, int first, double* jr, double* ji) {
    uint32_t r[4 * N];
    tmem_load<4 * N>(addr(base, owner) + 4 * first, r);
#pragma unroll
    for (int f = 0; f < N; ++f) {
      jr[f] = __hiloint2double(r[4 * f + 1], r[4 * f]);
      ji[f] = __hiloint2double(r[4 * f + 3], r[4 * f + 2]);
    }
  }
};

// |M|^2 of the 8 events whose momenta sit at the head of each event slice ([n_ext][4]).  Returns, on every lane of
// warp w < 8, the helicity- and colour-summed, averaged value of event w.  hel_out (optional, global [N_HEL], per warp)
// receives each helicity combination's share.  tmem: base address of the CTA's tensor-memory allocation.
template <class P> __device__ __forceinline__ double cta_me2_chunked(double* smem, double mass, double scale, double* hel_out, uint32_t tmem);

template <class P>
__device__ __forceinline__ double cta_me2(double* smem, double mass, double scale, double* hel_out, uint32_t tmem) {
  if constexpr (P::CHUNKED) {
    return cta_me2_chunked<P>(smem, mass, scale, hel_out, tmem);
  } else {
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  constexpr int W = P::W_EVENTS;
  constexpr bool SPLIT = P::SPLIT_J;
  static_assert(!SPLIT || P::N_WARPS == 2 * W, "two warps per event");
  // the warp index through a shuffle: the compiler then knows it is warp-uniform, so the item loop (table reads, op
  // and coefficient decoding, branches) runs on the uniform datapath
  const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int ev_w = warp & (W - 1), role = warp / W;   // dot stages: this warp's event, and which half of the flows
  // a5: subset momenta / denominators and external wavefunctions, work = (subset or leg, event)
  {
    const int t = threadIdx.x, ev = t % W;
    double* mom_s = smem + ev * STRIDE;
    me_phase0(t / W, 32 * P::N_WARPS / W, mom_s + 4 * P::N_EXT, mom_s, P::N_EXT, P::N_SUB, d_masks, d_kind, d_massive, d_extoff, mass);
  }
  __syncthreads();
  double* base = smem + 4 * P::N_EXT;  // event e's scratch = base + e * STRIDE
  static_assert(P::N_HEL_EVAL <= 32, "one helicity combination per lane");
  static_assert(P::N_PASS == 1 && P::W_EVENTS * P::VPI == 32, "the register-resident form evaluates the event in one pass");
  constexpr int NFW = JPark<P>::NFW;
  double jr[NFW], ji[NFW];
  const double* my = base + ev_w * STRIDE;
  double* sm_e = base + (lane % W) * STRIDE;   // items: lane = local variant j x event
  const int j = lane / W;
  const bool dot_warp = SPLIT || P::N_WARPS == W || warp < W;   // helper warps (if any) only run items
  int it = 0;
  // ONE copy of the item interpreter and one of each round's dot products in the instruction stream.  Warp w runs
  // items w, w + N_WARPS, ... of a stage: the generator balanced them by cost (a shared work counter was measured
  // and lost 4 %, profiles/r2_me_eval_summary.md).
  if constexpr (P::PIPELINED) {
    // Stage p = the items of one round + the dot products of the round before it (they read the other round region).
    // Warps 0-3 (one per scheduler) take the dot products first, warps 4-7 the items first, so that a scheduler mostly
    // holds one warp in a latency-bound item and one in a pipe-bound dot stage.  One copy of each in the instruction stream.
    static_assert(!SPLIT && P::N_WARPS == W && JPark<P>::ON, "pipelined form: eight warps, J parked in tensor memory");
    const bool group_a = warp < W / 2;
#pragma unroll 1
    for (int p = 0; p < P::N_STAGES; ++p) {
      const int end = P::stage_end(p), r = P::stage_dots(p);
#pragma unroll 1
      for (int ph = 0; ph < 2; ++ph) {
        const bool want_dots = r >= 0 && ((ph == 0) == group_a);
        const bool want_items = r < 0 ? ph == 0 : ((ph == 0) != group_a);
        if (want_dots) {
          if (r == 0) {
#pragma unroll
            for (int f = 0; f < NFW; ++f) { jr[f] = 0.0; ji[f] = 0.0; }
          } else {
            JPark<P>::template load<NFW>(tmem, warp, 0, jr, ji);
          }
          if (lane < P::N_HEL_EVAL) P::dots(r, my, lane, jr, ji);
          if (r + 1 < P::N_ROUNDS) JPark<P>::park(tmem, warp, jr, ji);
        }
        if (want_items) {
#pragma unroll 1
          for (int i = it + warp; i < end; i += P::N_WARPS) me_run_item<MADME_PREFETCH, P::VPI, P::NSLOT>(c_items[i], c_members, j, sm_e, mass);
        }
      }
      it = end;
      if (p + 1 < P::N_STAGES) __syncthreads();
    }
  } else {
#pragma unroll 1
  for (int p = 0; p < P::N_STAGES; ++p) {
    const int end = P::stage_end(p);
#pragma unroll 1
    for (int i = it + warp; i < end; i += P::N_WARPS) me_run_item<MADME_PREFETCH, P::VPI, P::NSLOT>(c_items[i], c_members, j, sm_e, mass);
    it = end;
    __syncthreads();
    const int r = P::stage_dots(p);
    if (r >= 0) {
      // J is defined here on every path (zero in the first round, un-parked afterwards): dead during the items
      if (dot_warp) {
        if (r == 0) {
#pragma unroll
          for (int f = 0; f < NFW; ++f) { jr[f] = 0.0; ji[f] = 0.0; }
        } else if (JPark<P>::ON) {
          JPark<P>::template load<NFW>(tmem, warp, 0, jr, ji);
        }
        if (lane < P::N_HEL_EVAL) {
          if (!SPLIT) P::dots(r, my, lane, jr, ji);
          else if (role == 0) P::dots_a(r, my, lane, jr, ji);
          else P::dots_b(r, my, lane, jr, ji);
        }
        if (JPark<P>::ON && (SPLIT || r + 1 < P::N_ROUNDS)) JPark<P>::park(tmem, warp, jr, ji);
      }
      if (r + 1 < P::N_ROUNDS) __syncthreads();   // the next round's items overwrite the round region
    }
  }
  }
  double v = 0.0;
  if (!SPLIT) {
    if (P::N_WARPS > W && warp >= W) return 0.0;
    if (lane < P::N_HEL_EVAL) v = P::colour(jr, ji);
  } else {
    // a9 with two warps per event: both halves are parked; role A contracts (A, A) and A x (first chunk of B), role B
    // (B, B) and (rest of B) x A read in two chunks; the two partial sums meet in shared memory
    __shared__ double v_b[W][32];
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (role == 0) {
      v = P::colour_own_a(jr, ji);
      if constexpr (P::CHUNK_B > 0) {
        double pr[P::CHUNK_B], pi[P::CHUNK_B];
        JPark<P>::template load<P::CHUNK_B>(tmem, warp + W, 0, pr, pi);
        v += P::colour_cross_a(jr, ji, pr, pi);
      }
    } else if constexpr (P::N_FLOW_B > 0) {
      v = P::colour_own_b(jr, ji);
      if constexpr (P::N_FLOW_B > P::CHUNK_B) {
        {
          double pr[P::CHUNK_A], pi[P::CHUNK_A];
          JPark<P>::template load<P::CHUNK_A>(tmem, warp - W, 0, pr, pi);
          v += P::colour_cross_b0(jr, ji, pr, pi);
        }
        if constexpr (P::N_FLOW_A > P::CHUNK_A) {
          double pr[P::N_FLOW_A - P::CHUNK_A], pi[P::N_FLOW_A - P::CHUNK_A];
          JPark<P>::template load<P::N_FLOW_A - P::CHUNK_A>(tmem, warp - W, P::CHUNK_A, pr, pi);
          v += P::colour_cross_b1(jr, ji, pr, pi);
        }
      }
    }
    if (lane >= P::N_HEL_EVAL) v = 0.0;
    if (role == 1) v_b[ev_w][lane] = v;
    __syncthreads();
    if (role == 1) return 0.0;
    v += v_b[ev_w][lane];
  }
  if (hel_out && lane < P::N_HEL_EVAL) {  // full index: leg 0 at +1 is bit 0; the parity partner has every helicity flipped
    const int hf = (lane << 1) | 1;
    hel_out[hf] = v * scale;
    hel_out[(P::N_HEL - 1) ^ hf] = v * scale;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return 2.0 * v * scale;
  }
}

// The form with the colour-flow vector in TENSOR MEMORY (P::CHUNKED).  For processes whose J does not fit a lane's registers
// (g g -> t tbar g g g: 120 flows), and for CTAs with more warps than events, where no warp can afford
// to keep J in registers.  The event is evaluated in P::N_PASS passes with the helicities of the frozen legs fixed, so that
// a lane holds one helicity combination; J of a pass occupies 4 N_FLOW 32-bit columns of 32 tensor-memory lanes per event
// (event e: lanes 32 (e % 4).., column block e / 4).  The unit of work of the dot stages is (event, chunk of P::CHUNK flows):
// load the chunk, add the round's dot products that feed it, store it back; of the colour stage (event, pair of chunks).
// A warp reaches only the lanes of its own sub-partition (warp % 4), so the N_WARPS / 4 warps of a sub-partition share the
// units of its W_EVENTS / 4 events.
// Items: the 32 lanes are W_EVENTS events x VPI helicity variants.
template <class P> struct ChunkIO {
  static constexpr int CH = P::CHUNK;
  static __device__ __forceinline__ void load(uint32_t taddr, double* jr, double* ji) {
    uint32_t q[4 * CH];
    tmem_load<4 * CH>(taddr, q);
#pragma unroll
    for (int f = 0; f < CH; ++f) { jr[f] = __hiloint2double(q[4 * f + 1], q[4 * f]); ji[f] = __hiloint2double(q[4 * f + 3], q[4 * f + 2]); }
  }
  static __device__ __forceinline__ void store(uint32_t taddr, const double* jr, const double* ji) {
    uint32_t q[4 * CH];
#pragma unroll
    for (int f = 0; f < CH; ++f) {
      q[4 * f] = __double2loint(jr[f]); q[4 * f + 1] = __double2hiint(jr[f]);
      q[4 * f + 2] = __double2loint(ji[f]); q[4 * f + 3] = __double2hiint(ji[f]);
    }
    tmem_store<4 * CH>(taddr, q);
  }
};

template <class P>
__device__ __forceinline__ double cta_me2_chunked(double* smem, double mass, double scale, double* hel_out, uint32_t tmem) {
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  constexpr int W = P::W_EVENTS, VPI = P::VPI, CH = P::CHUNK, NC = P::N_CHUNK, NW = P::N_WARPS;
  constexpr int EG = (W + 3) / 4, WG = NW / 4;   // events and warps per tensor-memory sub-partition
  constexpr int NPAIR = NC * (NC + 1) / 2;
  static_assert(W * VPI == 32 && (W == 4 || W == 8) && NW % 4 == 0 && P::N_HEL_EVAL <= 32 && EG * 4 * CH * NC <= 512, "geometry");
  __shared__ double v_part[WG][W][32];
  const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  double* base = smem + 4 * P::N_EXT;
  // items: eight events -> the lanes of a quarter warp are eight events (their stride is 16 B mod 128 B: no bank
  // conflict); four events -> the eight lanes of an event read one 128-byte line
  double* sm_e = base + (VPI == 4 ? lane % W : lane / VPI) * STRIDE;
  const int j = VPI == 4 ? lane / W : lane % VPI;
  const int sub = warp & 3, k_w = warp >> 2;
  const uint32_t tsub = tmem + (static_cast<uint32_t>(32 * sub) << 16);   // this sub-partition's lanes, column 0
  double v = 0.0;
#pragma unroll 1
  for (int pass = 0; pass < P::N_PASS; ++pass) {
    {
      const int t = threadIdx.x, ev = t % W;
      double* mom_s = smem + ev * STRIDE;
      me_phase0(t / W, 32 * NW / W, mom_s + 4 * P::N_EXT, mom_s, P::N_EXT, P::N_SUB, d_masks, d_kind, d_massive, d_extoff, mass,
                P::FROZEN_MASK, P::frozen_helicities(pass));
    }
    {   // J = 0
      double zr[CH], zi[CH];
#pragma unroll
      for (int f = 0; f < CH; ++f) { zr[f] = 0.0; zi[f] = 0.0; }
#pragma unroll 1
      for (int u = k_w; u < EG * NC; u += WG) ChunkIO<P>::store(tsub + (u / NC) * 4 * CH * NC + 4 * CH * (u % NC), zr, zi);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    int it = 0;
#pragma unroll 1
    for (int p = 0; p < P::N_STAGES; ++p) {
      const int end = P::stage_end(p);
#pragma unroll 1
      for (int i = it + warp; i < end; i += NW) me_run_item<MADME_PREFETCH_CHUNKED, VPI, P::NSLOT>(c_items[i], c_members, j, sm_e, mass);
      it = end;
      __syncthreads();
      const int r = P::stage_dots(p);
      if (r >= 0) {
        // the (event, chunk) units of this sub-partition that the round feeds, dealt to its warps by cost (generator)
#pragma unroll 1
        for (int u = 0; u < EG * NC; ++u) {
          const int ei = u / NC, c = u % NC;
          if (!P::has_dots(r, c)) continue;
          if ((P::dot_owner(r, c) + ei) % WG != k_w) continue;
          if (4 * ei + sub >= W) continue;
          const uint32_t ta = tsub + ei * 4 * CH * NC + 4 * CH * c;
          double jr[CH], ji[CH];
          ChunkIO<P>::load(ta, jr, ji);
          if (lane < P::N_HEL_EVAL) P::dots(r, c, base + (4 * ei + sub) * STRIDE, lane, jr, ji);
          ChunkIO<P>::store(ta, jr, ji);
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();   // the next round's items (or the next pass) overwrite the round region; J is complete
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      }
    }
    // a9, a10: J^dagger CF J over (event, pair of chunks) units; this pass's helicities
    double vp[EG];
#pragma unroll
    for (int ei = 0; ei < EG; ++ei) vp[ei] = 0.0;
#pragma unroll 1
    for (int u = k_w; u < EG * NPAIR; u += WG) {
      const int ei = u / NPAIR;
      int q = u % NPAIR, ca = 0;
      while (q >= NC - ca) { q -= NC - ca; ++ca; }
      const int cb = ca + q;
      double ar[CH], ai[CH], t;
      ChunkIO<P>::load(tsub + ei * 4 * CH * NC + 4 * CH * ca, ar, ai);
      if (cb == ca) {
        t = P::colour_diag(ca, ar, ai);
      } else {
        double br[CH], bi[CH];
        ChunkIO<P>::load(tsub + ei * 4 * CH * NC + 4 * CH * cb, br, bi);
        t = P::colour_pair(ca, cb, ar, ai, br, bi);
      }
#pragma unroll
      for (int e2 = 0; e2 < EG; ++e2) vp[e2] += (e2 == ei) ? t : 0.0;
    }
#pragma unroll
    for (int ei = 0; ei < EG; ++ei)
      if (4 * ei + sub < W) v_part[k_w][4 * ei + sub][lane] = (lane < P::N_HEL_EVAL) ? vp[ei] : 0.0;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (warp < W) {
      double t = 0.0;
#pragma unroll
      for (int k = 0; k < WG; ++k) t += v_part[k][warp][lane];
      if (hel_out && lane < P::N_HEL_EVAL) {   // the parity partner has every helicity flipped
        const int hf = P::full_helicity(lane, pass);
        hel_out[hf] = t * scale;
        hel_out[(P::N_HEL - 1) ^ hf] = t * scale;
      }
      v += t;
    }
    if (pass + 1 < P::N_PASS) __syncthreads();   // v_part is rewritten by the next pass
  }
  if (warp >= W) return 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return 2.0 * v * scale;
}

// W_EVENTS events per CTA (blockDim.x = 32 P::N_WARPS); persistent grid, batches of W_EVENTS consecutive events.
template <class P>
__global__ void __launch_bounds__(32 * P::N_WARPS, 1) me_eval_kernel(const double* __restrict__ momenta, double* __restrict__ me2,
                                                              double* __restrict__ me2_hel, long long n_ev, double mass, double scale) {
  extern __shared__ __align__(16) double smem[];
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  constexpr int W = P::W_EVENTS;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t tmem = JPark<P>::ON ? tmem_alloc<JPark<P>::COLS>() : 0u;
  const long long n_batches = (n_ev + W - 1) / W;
  // (not for the chunked processes: their shared memory is full and a batch takes millions of cycles)
  constexpr bool PRE = MADME_PREFETCH_MOMENTA && !P::CHUNKED;
  // The momenta of the NEXT batch travel from HBM into a small staging buffer (cp.async, one double per thread) while this
  // batch is computed: the DRAM latency at the head of a batch was 2.7 % of the kernel's samples (7 % for the small
  // processes).  Every thread copies, waits for and reads its own element, so no barrier is involved.
  __shared__ __align__(16) double next_mom[PRE ? W : 1][PRE ? 4 * P::N_EXT : 2];
  const bool loader = (P::N_WARPS == W || warp < W) && lane < 4 * P::N_EXT;
  auto prefetch = [&](long long b) {
    if (PRE && loader) {
      const long long ev = min(b * W + (warp & (W - 1)), n_ev - 1);   // events past the end repeat the last one
      const unsigned dst = static_cast<unsigned>(__cvta_generic_to_shared(&next_mom[warp][lane]));
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(dst), "l"(momenta + ev * (4 * P::N_EXT) + lane) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  if (PRE && static_cast<long long>(blockIdx.x) < n_batches) prefetch(blockIdx.x);
  for (long long b = blockIdx.x; b < n_batches; b += gridDim.x) {
    // events past the end repeat the last one (computed, not stored)
    const long long ev = min(b * W + (warp & (W - 1)), n_ev - 1);
    if constexpr (PRE) {
      asm volatile("cp.async.wait_all;" ::: "memory");
      if (loader) smem[warp * STRIDE + lane] = next_mom[warp][lane];
      if (b + gridDim.x < n_batches) prefetch(b + gridDim.x);
    } else {
      if (loader) smem[warp * STRIDE + lane] = momenta[ev * (4 * P::N_EXT) + lane];
    }
    __syncthreads();
    const double r = cta_me2<P>(smem, mass, scale, (me2_hel && b * W + (warp & (W - 1)) < n_ev) ? me2_hel + ev * P::N_HEL : nullptr, tmem);
    if ((P::N_WARPS == W || warp < W) && lane == 0 && me2 && b * W + warp < n_ev) me2[ev] = r;
    __syncthreads();
  }
  if (JPark<P>::ON) tmem_free<JPark<P>::COLS>(tmem);
}

}  // namespace madme
