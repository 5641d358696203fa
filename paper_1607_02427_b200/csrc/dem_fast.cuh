// dem_fast.cuh -- the FP32 pair-feature kernel of libdem_b200 for sm_100a: packed contact search + cooperative
// evaluation of the candidate terms.  (The generic k_pair of dem_kernels.cuh stays as the FP64 path.)
//
// The paper fuses the nearest-point search and the potential in one kernel and names the resulting register
// pressure as its bottleneck, with "split contact search from force evaluation" as future work.  On
// B200 the search is bound by FP32 issue slots, so it is written here with Blackwell's packed FP32 instructions
// (FFMA2 / FADD2 / FMUL2, PTX fma.rn.f32x2): one lane carries TWO outer features of particle j in the halves of
// 64-bit registers and sweeps them over the inner features of particle i, which it reads as warp-uniform shared-memory
// broadcasts (FFMA2 takes a 32-bit register as a broadcast operand).  A packed instruction occupies the FMA pipe
// for two cycles but takes ONE issue slot, which leaves the slots the clamps, minima, shared-memory loads and loop
// control need (measured on B200: 8 FFMA2 + 8 FMNMX per 17.8 cycles against 8 FFMA + 4 FMNMX per 12.5).
//
//   search  : every Eq. 1 / Eq. 2 term gets its nearest-point distance r*^2
//             from a branch-free packed formulation; the only output is one bit per packed evaluation,
//             "some r*^2 < rc_search^2", shifted into a per-lane mask (sign bit of r^2 - rc_search^2, funnel shift).
//   queue   : after each sweep the lanes of a warp append their flagged (outer, inner) term ids to a warp-private
//             shared-memory queue (ballot ranks: deterministic order, no atomics).
//   evaluate: whenever 32 candidates are queued the warp evaluates them TOGETHER, one term per lane, with the exact
//             scalar routines of dem_math.cuh (parallel-edge rule R5, WCA, force, torque), and hands each
//             contribution back to the lane that owns the pair with warp shuffles, in queue order.  Contact terms
//             therefore cost one lane-evaluation each instead of one divergent warp-evaluation each.
//
// rc_search is the WCA cutoff plus a slack that covers FP32 rounding of the packed formulation and the error of its
// segment-segment routine on near-parallel edges, so every term the scalar routine finds inside
// the cutoff is a candidate; the scalar routine alone decides what contributes.
#pragma once
#include "dem_kernels.cuh"

namespace dem {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pk(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 bc(float x) { return pk(x, x); }  // ptxas folds this into FFMA2's .F32 broadcast operand
__device__ __forceinline__ u64 neg2(u64 v) {                     // folded into the operand's negate modifier
    float lo, hi;
    upk(v, lo, hi);
    return pk(-lo, -hi);
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float mul_sat(float a, float b) {
    float r;
    asm("mul.rn.sat.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
    return r;
}
// shift the sign bit of v into the mask: bit set <=> v < 0
__device__ __forceinline__ unsigned push_sign(unsigned mask, float v) { return __funnelshift_l(__float_as_uint(v), mask, 1); }

#define DEM_QCAP 96        // 31 left over + at most 64 appended per round
#define DEM_Q_INVALID 0xffffffffu
enum { PH_EE = 0, PH_VF_OWN = 1, PH_VF_OTHER = 2, PH_VE_OWN = 3, PH_VE_OTHER = 4, PH_VF_BOTH = 5 /* sweeps only */ };

// what the cooperative evaluation needs, kept in shared memory (the hot loops hold their own copies in registers)
struct FastShared {
    ShapeView<float> A, B;
    PairConst<float> pc;
};

// candidate entry: owner slot (6 bits: up to 64 pairs per warp tile) | phase (3) | outer feature (11) | inner feature (12)
__device__ __forceinline__ unsigned q_entry(int owner, int phase, int outer, int inner) {
    return ((unsigned)owner << 26) | ((unsigned)phase << 23) | ((unsigned)outer << 12) | (unsigned)inner;
}

// ---- evaluate: up to 32 queued candidates, one per lane -----------------------------------------------------------------
// q: this warp's queue (qn entries, the first cnt <= 32 are consumed and the rest moved to the front); sacc: this warp's
// per-lane accumulators [7][32] = (F.xyz, T.xyz, u) in the owner's body frame; scnt: this warp's counters (active,
// degenerate, parallel).  sp: the warp's staged pose records [3][nown] (plane-major, indexed by owner lane); the
// evaluating lane reads its owner's pose from there.
// Contributions are added to the owner in queue order, so the result does not depend on scheduling.  Returns, per lane,
// which of its owner slots received a contribution (only those pairs get a result record).
static __device__ __noinline__ unsigned drain_terms(const FastShared* fs, unsigned* q, float* sacc, unsigned* scnt, int cnt,
                                                    int qn, const f4* sp, int nown) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    DEM_ASSERT(cnt >= 0 && cnt <= 32 && cnt <= qn && qn <= DEM_QCAP);
    const unsigned e = lane < cnt ? q[lane] : DEM_Q_INVALID;
    const int rem = qn - cnt;
    const unsigned v0 = lane < rem ? q[cnt + lane] : 0u, v1 = lane + 32 < rem ? q[cnt + 32 + lane] : 0u;
    __syncwarp();
    if (lane < rem) q[lane] = v0;
    if (lane + 32 < rem) q[32 + lane] = v1;
    __syncwarp();
    const int owner = e == DEM_Q_INVALID ? lane : (int)(e >> 26);
    DEM_ASSERT(owner >= 0 && owner < nown);
    float R[9], t[3];
    {
        const f4 p0 = sp[owner], p1 = sp[nown + owner], p2 = sp[2 * nown + owner];
        R[0] = p0.x; R[1] = p0.y; R[2] = p0.z; R[3] = p0.w; R[4] = p1.x; R[5] = p1.y; R[6] = p1.z; R[7] = p1.w;
        R[8] = p2.x; t[0] = p2.y; t[1] = p2.z; t[2] = p2.w;
    }
    PairAcc<float> loc;
    loc.F[0] = loc.F[1] = loc.F[2] = loc.T[0] = loc.T[1] = loc.T[2] = loc.u = 0.f;
    loc.nactive = loc.ndegen = loc.npar = 0u;
    if (e != DEM_Q_INVALID) {
        const int phase = (int)((e >> 23) & 7u), o = (int)((e >> 12) & 0x7ffu), k = (int)(e & 0xfffu);
        const ShapeView<float> A = fs->A, B = fs->B;
        DEM_ASSERT(phase == PH_EE ? (o < B.ne && k < A.ne)
                   : phase == PH_VF_OWN ? (o < B.nv && k < A.nf)
                   : phase == PH_VF_OTHER ? (o < A.nv && k < B.nf)
                   : phase == PH_VE_OWN ? (o < B.nv && k < A.ne) : (phase == PH_VE_OTHER && o < A.nv && k < B.ne));
        const PairConst<float> pc = fs->pc;
        float p[3];
        // The 3D kinds share one copy of the face routines and one of the WCA code (the kernel's code has to stay small:
        // DESIGN.md section 10): each kind leaves ci (interaction point on i), del = c_i - c_j, r2; then one accumulate.
        if (phase <= PH_VF_OTHER) {
            float ci[3], del[3], r2 = 0.f;
            bool hit, par = false;
            if (phase == PH_EE) {
                float d2[3], ee, inv_e;
                edge_to_i<float>(B, o, R, t, p, d2, ee, inv_e);
                hit = term_ee_geom<float>(A, k, p[0], p[1], p[2], d2[0], d2[1], d2[2], ee, inv_e, pc, ci, del, r2, par);
            } else {
                const bool own = phase == PH_VF_OWN;  // vertex of j against a face of i (i's frame) / of i against j (j's)
                const ShapeView<float>& S = own ? A : B;
                const f4 v = own ? B.V[o] : A.V[o];
                if (own) vertex_to_i<float>(v.x, v.y, v.z, R, t, p);
                else vertex_to_j<float>(v.x, v.y, v.z, R, t, p);
                r2 = point_face_r2<float>(S, k, p[0], p[1], p[2]);
                hit = r2 < pc.rc2;
                if (hit) {
                    float dx, dy, dz;  // p - c with c on the face
                    point_face_del<float>(S, k, p[0], p[1], p[2], dx, dy, dz);
                    if (own) {  // c_i = c, c_j = p: del = -(p - c)      (term_vf_own)
                        ci[0] = p[0] - dx; ci[1] = p[1] - dy; ci[2] = p[2] - dz;
                        del[0] = -dx; del[1] = -dy; del[2] = -dz;
                    } else {    // c_i = the vertex, del = R (p' - c')      (term_vf_other)
                        ci[0] = v.x; ci[1] = v.y; ci[2] = v.z;
                        del[0] = R[0] * dx + R[1] * dy + R[2] * dz;
                        del[1] = R[3] * dx + R[4] * dy + R[5] * dz;
                        del[2] = R[6] * dx + R[7] * dy + R[8] * dz;
                    }
                }
            }
            if (hit) wca_accumulate<float>(pc, loc, ci[0], ci[1], ci[2], del[0], del[1], del[2], r2, par);
        } else if (phase == PH_VE_OWN) {
            const f4 v = B.V[o];
            vertex_to_i<float>(v.x, v.y, 0.f, R, t, p);
            term_ve_own<float>(A, k, p[0], p[1], pc, loc);
        } else {
            const f4 v = A.V[o];
            vertex_to_j<float>(v.x, v.y, 0.f, R, t, p);
            term_ve_other<float>(B, k, v.x, v.y, p[0], p[1], R, pc, loc);
        }
    }
    const unsigned na = __reduce_add_sync(full, loc.nactive), nd = __reduce_add_sync(full, loc.ndegen),
                   np = __reduce_add_sync(full, loc.npar);
    if (lane == 0) {
        scnt[0] += na;
        scnt[1] += nd;
        scnt[2] += np;
    }
    // Add the lanes' results to their owners' accumulators.  Lanes with different owners write different shared-memory
    // words, so they go together; lanes with the same owner take turns in lane order (round r: the lane that is the
    // r-th of its owner's lanes), which is the order a serial walk over the lanes would give: the sums do not depend on
    // scheduling, bit for bit.
    const bool actl = loc.nactive != 0u;
    const unsigned peers = __match_any_sync(full, actl ? owner : 64 + lane);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    const int rounds = (int)__reduce_max_sync(full, actl ? (unsigned)rank + 1u : 0u);
    for (int r = 0; r < rounds; ++r) {
        if (actl && rank == r) {
            sacc[0 * nown + owner] += loc.F[0]; sacc[1 * nown + owner] += loc.F[1]; sacc[2 * nown + owner] += loc.F[2];
            sacc[3 * nown + owner] += loc.T[0]; sacc[4 * nown + owner] += loc.T[1]; sacc[5 * nown + owner] += loc.T[2];
            sacc[6 * nown + owner] += loc.u;
        }
        __syncwarp();
    }
    // bit h of the result: this lane's owner slot lane + 32 h received a contribution
    const unsigned w0 = __reduce_or_sync(full, actl && owner < 32 ? 1u << owner : 0u);
    const unsigned w1 = nown > 32 ? __reduce_or_sync(full, actl && owner >= 32 ? 1u << (owner - 32) : 0u) : 0u;
    const unsigned touched = ((w0 >> lane) & 1u) | (((w1 >> lane) & 1u) << 1);
    __syncwarp();
    return touched;
}

// per-warp state of the search loops
struct WarpCtx {
    const FastShared* fs;
    unsigned* q;
    float* sacc;
    unsigned* scnt;
    int qn;    // queued candidates (warp-uniform)
    int lane;
    const f4* sp;  // staged pose records of the current tile, [3][nown] (R, t)
    int nown;      // pairs per warp tile: 32 (k_pair_fast) or 64 (k_pair_cull)
    unsigned touched;  // bit h: owner slot lane + 32 h of this lane has received a contribution in the current tile
};

// ---- queue: append the candidates flagged in mask[] and evaluate while a full warp of them is waiting ------------------
// mask bit (n - 1 - i) <=> the packed evaluation of inner feature k0 + i flagged a candidate in either half: both
// terms are queued (the scalar routine sorts them out).  The halves belong to (owner lane, outer feature) = (wa, oa)
// and (wb, ob); ok_a / ok_b say whether the half holds a real feature (tiles and item lists are padded).
__device__ __forceinline__ void push_one(WarpCtx& w, int phase_a, int phase_b, unsigned m, int n, int k0, int wa, int oa,
                                         bool ok_a, int wb, int ob, bool ok_b) {
    const unsigned full = 0xffffffffu;
    const unsigned lt = (1u << w.lane) - 1u;
    while (__any_sync(full, m != 0u)) {
        const bool have = m != 0u;
        const int bit = 31 - __clz((int)m);
        const int k = k0 + (n - 1 - bit);
        if (have) m &= ~(1u << bit);
        const bool ha = have && ok_a, hb = have && ok_b;
        const unsigned ba = __ballot_sync(full, ha), bb = __ballot_sync(full, hb);
        const int na = __popc(ba);
        DEM_ASSERT(w.qn >= 0 && w.qn + na + __popc(bb) <= DEM_QCAP);
        if (ha) w.q[w.qn + __popc(ba & lt)] = q_entry(wa, phase_a, oa, k);
        if (hb) w.q[w.qn + na + __popc(bb & lt)] = q_entry(wb, phase_b, ob, k);
        w.qn += na + __popc(bb);
        __syncwarp();
        while (w.qn >= 32) {
            w.touched |= drain_terms(w.fs, w.q, w.sacc, w.scnt, 32, w.qn, w.sp, w.nown);
            w.qn -= 32;
        }
    }
}

// the same for ONE inner feature per lane (k may differ from lane to lane; `have` = this lane flagged a candidate)
__device__ __forceinline__ void push_lane(WarpCtx& w, int phase_a, int phase_b, bool have, int k, int wa, int oa, bool ok_a,
                                          int wb, int ob, bool ok_b) {
    const unsigned full = 0xffffffffu;
    const unsigned lt = (1u << w.lane) - 1u;
    const bool ha = have && ok_a, hb = have && ok_b;
    const unsigned ba = __ballot_sync(full, ha), bb = __ballot_sync(full, hb);
    if ((ba | bb) == 0u) return;
    const int na = __popc(ba);
    DEM_ASSERT(w.qn >= 0 && w.qn + na + __popc(bb) <= DEM_QCAP);
    if (ha) w.q[w.qn + __popc(ba & lt)] = q_entry(wa, phase_a, oa, k);
    if (hb) w.q[w.qn + na + __popc(bb & lt)] = q_entry(wb, phase_b, ob, k);
    w.qn += na + __popc(bb);
    __syncwarp();
    while (w.qn >= 32) {
        w.touched |= drain_terms(w.fs, w.q, w.sacc, w.scnt, 32, w.qn, w.sp, w.nown);
        w.qn -= 32;
    }
}

// tile form: lane-owned outer features o0 + 2 tau and o0 + 2 tau + 1
template <int T>
__device__ __forceinline__ void push_and_drain(WarpCtx& w, int phase, const unsigned (&mask)[T], int n, int k0, int o0,
                                               int o_end) {
    // one copy of the queue code per call site, not one per packed pair (code size: DESIGN.md section 10); the mask of
    // the pair is picked with selects so that the array stays in registers
    static_assert(T <= 3, "mask select below");
#pragma unroll 1
    for (int tau = 0; tau < T; ++tau) {
        const unsigned m = tau == 0 ? mask[0] : (tau == 1 || T < 3) ? mask[T > 1 ? 1 : 0] : mask[T > 2 ? 2 : 0];
        push_one(w, phase, phase, m, n, k0, w.lane, o0 + 2 * tau, o0 + 2 * tau < o_end, w.lane, o0 + 2 * tau + 1,
                 o0 + 2 * tau + 1 < o_end);
    }
}

// ---- search: packed nearest-point distances ---------------------------------------------------------------------------
// Segment-segment (first sum of Eq. 1): inner edge of i as scalars e0 = (p1, |d1|^2), e1 = (d1, 1/|d1|^2), parameter
// s in [0,1]; two outer edges of j packed, unit directions d2, parameter t in [0, L2] (length units), np2 = -p2.
// Closest points of the two lines from the normal equations, then the textbook clamp cascade with the second clamp of
// s taken unconditionally (KKT: when t was not clamped it reproduces s).  Returns min over the two halves of
// r^2 - rc_search^2.  Near-parallel edges (|d1 x d2|^2 -> 0) make s inaccurate but never out of [0,1], and t, s2 are
// then exact for that s, so r is off by at most sin(angle) x edge length: covered by rc_search's slack.
__device__ __forceinline__ float ee_eval(const f4 e0, const f4 e1, u64 np2x, u64 np2y, u64 np2z, u64 d2x, u64 d2y,
                                         u64 d2z, u64 g, float Llo, float Lhi, float nrc2) {
    const u64 rx = add2(bc(e0.x), np2x), ry = add2(bc(e0.y), np2y), rz = add2(bc(e0.z), np2z);  // r = p1 - p2
    const u64 b = fma2(bc(e1.z), d2z, fma2(bc(e1.y), d2y, mul2(bc(e1.x), d2x)));              // d1 . d2
    const u64 c = fma2(bc(e1.z), rz, fma2(bc(e1.y), ry, mul2(bc(e1.x), rx)));                 // d1 . r
    // d2 . r = d2 . p1 + g with g = -d2 . p2 per outer edge: keeps one operand of every FFMA2 a broadcast scalar
    // (three 64-bit register operands cost the register file a third cycle)
    const u64 f = fma2(d2z, bc(e0.z), fma2(d2y, bc(e0.y), fma2(d2x, bc(e0.x), g)));
    const u64 nn = fma2(neg2(b), b, bc(e0.w));                                                // |d1|^2 - b^2
    const u64 num = fma2(b, f, neg2(c));
    float nl, nh, ul, uh;
    upk(nn, nl, nh);
    upk(num, ul, uh);
    const u64 s = pk(mul_sat(ul, rcp(nl)), mul_sat(uh, rcp(nh)));
    float xl, xh;
    upk(fma2(b, s, f), xl, xh);
    const u64 tt = pk(fminf(fmaxf(xl, 0.f), Llo), fminf(fmaxf(xh, 0.f), Lhi));
    float yl, yh;
    upk(fma2(b, tt, neg2(c)), yl, yh);
    const u64 s2 = pk(mul_sat(yl, e1.w), mul_sat(yh, e1.w)), ntt = neg2(tt);
    const u64 dx = fma2(ntt, d2x, fma2(s2, bc(e1.x), rx));
    const u64 dy = fma2(ntt, d2y, fma2(s2, bc(e1.y), ry));
    const u64 dz = fma2(ntt, d2z, fma2(s2, bc(e1.z), rz));
    float lo, hi;
    upk(fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, bc(nrc2)))), lo, hi);
    return fminf(lo, hi);
}

// One boundary edge (or 2D edge) e0 = (., ., ux, uy), e1 = (len, cs, cm, len/2) against two packed points (x, y):
// side = u x q + cs (>= 0 on the inner side), centred along-edge coordinate am = u . q + cm (0 at the edge's midpoint),
// excess = max(|am| - len/2, 0): the point's distance^2 from the segment is side^2 + excess^2.
__device__ __forceinline__ void edge2_eval(const f4 e0, const f4 e1, u64 x, u64 y, u64& side, u64& exc) {
    side = fma2(bc(e0.z), y, fma2(bc(-e0.w), x, bc(e1.y)));
    float am_l, am_h;
    upk(fma2(bc(e0.z), x, fma2(bc(e0.w), y, bc(e1.z))), am_l, am_h);
    exc = pk(fmaxf(fabsf(am_l) - e1.w, 0.f), fmaxf(fabsf(am_h) - e1.w, 0.f));
}

// minimum of n values with 3-input minima (FMNMX3)
template <int N> __device__ __forceinline__ float min_tree(const float (&v)[N]) {
    float r = v[0];
#pragma unroll
    for (int k = 1; k + 1 < N; k += 2) r = fminf(fminf(r, v[k]), v[k + 1]);
    if ((N & 1) == 0) r = fminf(r, v[N - 1]);
    return r;
}

// Point against closed convex polygon face (R1/R2): two packed points against face header F[0..2] and its M boundary
// edges.  r^2 = h^2 + (inside ? 0 : min over edges of side^2 + excess^2).  Updates mask[tau] for T packed point pairs.
template <int T, int M>
__device__ __forceinline__ void face_eval(const f4* __restrict__ F, const f4* __restrict__ FE, const u64 (&px)[T],
                                          const u64 (&py)[T], const u64 (&pz)[T], float nrc2, unsigned (&mask)[T]) {
    const f4 f0 = F[0], f1 = F[1], f2 = F[2];
    u64 x[T], y[T], hh[T];
    float sl[T][M], sh[T][M], dl[T][M], dh[T][M];
#pragma unroll
    for (int tau = 0; tau < T; ++tau) {
        x[tau] = fma2(bc(f0.z), pz[tau], fma2(bc(f0.y), py[tau], fma2(bc(f0.x), px[tau], bc(f0.w))));
        y[tau] = fma2(bc(f1.z), pz[tau], fma2(bc(f1.y), py[tau], fma2(bc(f1.x), px[tau], bc(f1.w))));
        const u64 h = fma2(bc(f2.z), pz[tau], fma2(bc(f2.y), py[tau], fma2(bc(f2.x), px[tau], bc(f2.w))));
        hh[tau] = fma2(h, h, bc(nrc2));
    }
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const f4 e0 = FE[2 * m], e1 = FE[2 * m + 1];
#pragma unroll
        for (int tau = 0; tau < T; ++tau) {
            u64 side, exc;
            edge2_eval(e0, e1, x[tau], y[tau], side, exc);
            upk(side, sl[tau][m], sh[tau][m]);
            upk(fma2(exc, exc, mul2(side, side)), dl[tau][m], dh[tau][m]);
        }
    }
#pragma unroll
    for (int tau = 0; tau < T; ++tau) {
        const u64 sel = pk(min_tree<M>(sl[tau]) >= 0.f ? 0.f : min_tree<M>(dl[tau]),
                           min_tree<M>(sh[tau]) >= 0.f ? 0.f : min_tree<M>(dh[tau]));
        float lo, hi;
        upk(add2(hh[tau], sel), lo, hi);
        mask[tau] = push_sign(mask[tau], fminf(lo, hi));
    }
}

// the same for any number of boundary edges (run-time loop)
template <int T>
__device__ __forceinline__ void face_eval_any(const f4* __restrict__ F, const f4* __restrict__ FE, int mcount,
                                              const u64 (&px)[T], const u64 (&py)[T], const u64 (&pz)[T], float nrc2,
                                              unsigned (&mask)[T]) {
    const f4 f0 = F[0], f1 = F[1], f2 = F[2];
    u64 x[T], y[T], hh[T];
    float smin_l[T], smin_h[T], dmin_l[T], dmin_h[T];
#pragma unroll
    for (int tau = 0; tau < T; ++tau) {
        x[tau] = fma2(bc(f0.z), pz[tau], fma2(bc(f0.y), py[tau], fma2(bc(f0.x), px[tau], bc(f0.w))));
        y[tau] = fma2(bc(f1.z), pz[tau], fma2(bc(f1.y), py[tau], fma2(bc(f1.x), px[tau], bc(f1.w))));
        const u64 h = fma2(bc(f2.z), pz[tau], fma2(bc(f2.y), py[tau], fma2(bc(f2.x), px[tau], bc(f2.w))));
        hh[tau] = fma2(h, h, bc(nrc2));
        smin_l[tau] = smin_h[tau] = dmin_l[tau] = dmin_h[tau] = 1e30f;
    }
    for (int m = 0; m < mcount; ++m) {
        const f4 e0 = FE[2 * m], e1 = FE[2 * m + 1];
#pragma unroll
        for (int tau = 0; tau < T; ++tau) {
            u64 side, exc;
            edge2_eval(e0, e1, x[tau], y[tau], side, exc);
            float sl, sh, dl, dh;
            upk(side, sl, sh);
            upk(fma2(exc, exc, mul2(side, side)), dl, dh);
            smin_l[tau] = fminf(smin_l[tau], sl);
            smin_h[tau] = fminf(smin_h[tau], sh);
            dmin_l[tau] = fminf(dmin_l[tau], dl);
            dmin_h[tau] = fminf(dmin_h[tau], dh);
        }
    }
#pragma unroll
    for (int tau = 0; tau < T; ++tau) {
        const u64 sel = pk(smin_l[tau] >= 0.f ? 0.f : dmin_l[tau], smin_h[tau] >= 0.f ? 0.f : dmin_h[tau]);
        float lo, hi;
        upk(add2(hh[tau], sel), lo, hi);
        mask[tau] = push_sign(mask[tau], fminf(lo, hi));
    }
}

// sweep T packed pairs of points over faces [f0, f1) of shape S (at most 32 faces: one mask bit each).  Faces are
// stored sorted by boundary-edge count; sd lists the runs, so the common sizes run unrolled without a per-face branch.
template <int T>
__device__ __forceinline__ void sweep_faces(const ShapeView<float>& S, const ShapeDev& sd, int f0, int f1,
                                            const u64 (&px)[T], const u64 (&py)[T], const u64 (&pz)[T], float nrc2,
                                            unsigned (&mask)[T]) {
    if (sd.grp_m[0] == 0) {  // too many different face sizes: read every face's header
        for (int f = f0; f < f1; ++f) {
            const f4 f3 = S.F[4 * f + 3];
            face_eval_any<T>(S.F + 4 * f, S.FE + 2 * (int)f3.x, (int)f3.y, px, py, pz, nrc2, mask);
        }
        return;
    }
    int fbase = 0, febase = 0;
#pragma unroll 1
    for (int g = 0; g < DEM_MAX_FACE_GROUPS && sd.grp_n[g] > 0; ++g) {
        const int m = sd.grp_m[g], fend = fbase + sd.grp_n[g];
        const int lo = max(f0, fbase), hi = min(f1, fend);
        if (lo < hi) {
            const f4* F = S.F + 4 * lo;
            const f4* FE = S.FE + 2 * (febase + (lo - fbase) * m);
            const int n = hi - lo;
            switch (m) {
                case 3:
                    for (int f = 0; f < n; ++f, F += 4, FE += 6) face_eval<T, 3>(F, FE, px, py, pz, nrc2, mask);
                    break;
                case 4:
                    for (int f = 0; f < n; ++f, F += 4, FE += 8) face_eval<T, 4>(F, FE, px, py, pz, nrc2, mask);
                    break;
                case 5:
                    for (int f = 0; f < n; ++f, F += 4, FE += 10) face_eval<T, 5>(F, FE, px, py, pz, nrc2, mask);
                    break;
                case 6:
                    for (int f = 0; f < n; ++f, F += 4, FE += 12) face_eval<T, 6>(F, FE, px, py, pz, nrc2, mask);
                    break;
                default:
                    for (int f = 0; f < n; ++f, F += 4, FE += 2 * m) face_eval_any<T>(F, FE, m, px, py, pz, nrc2, mask);
                    break;
            }
        }
        febase += sd.grp_n[g] * m;
        fbase = fend;
    }
}

// R_i (rounded once from FP64, as pair_pose does) and the minimum-image separation d of a pair, for the few pairs that
// contribute: the pose records hold only R and t (48 bytes per pair), and a contributing pair fetches its two particles
// again instead of every pair carrying another 48 bytes through k_pose.  The arithmetic is that of k_pose, bit for bit.
static __device__ __forceinline__ void pose_tail(const void* pos, const void* quat, int pos_double, const BoxDev box, int2 ij,
                                              float* Mi, float* dout) {
    d4 xi, xj, qi;
    if (pos_double) {
        xi = load4d(static_cast<const double*>(pos), ij.x);
        xj = load4d(static_cast<const double*>(pos), ij.y);
        qi = load4d(static_cast<const double*>(quat), ij.x);
    } else {
        xi = load4d(static_cast<const float*>(pos), ij.x);
        xj = load4d(static_cast<const float*>(pos), ij.y);
        qi = load4d(static_cast<const float*>(quat), ij.x);
    }
    double d[3] = {xj.x - xi.x, xj.y - xi.y, box.dim == 3 ? xj.z - xi.z : 0.0};
    d[0] -= box.L[0] * rint(d[0] * box.invL[0]);
    d[1] -= box.L[1] * rint(d[1] * box.invL[1]);
    if (box.dim == 3) d[2] -= box.L[2] * rint(d[2] * box.invL[2]);
    double Di[9];
    quat_to_mat<double>(qi.x, qi.y, qi.z, qi.w, Di);
#pragma unroll
    for (int k = 0; k < 9; ++k) Mi[k] = (float)Di[k];
    dout[0] = (float)d[0]; dout[1] = (float)d[1]; dout[2] = (float)d[2];
}

// ---- a3: relative pose of every pair of a class, compacted -----------------------------------------------------------
// One thread per unique pair: minimum-image separation d, exact reach test (R10), relative pose R = R_i^T R_j,
// t = R_i^T d and R_i in FP64, rounded once to float.  Pairs inside the reach are compacted into the
// class's work list (block slices padded to whole warps: see below); pairs beyond it get their result-record flag cleared
// here (nothing is written for them, the reduction skips them) and never reach the search kernel, so its warps carry 32
// live pairs each.  Pose record, plane-major for coalesced loads: [3][npairs] float4 =
// (R0 R1 R2 R3) (R4 R5 R6 R7) (R8 t0 t1 t2); pidx[c] = the pair's index.  (R_i and d, which only a contributing pair
// needs, are recomputed by that pair: pose_tail.)
template <typename PosT, int DIM> __global__ void __launch_bounds__(DEM_POSE_THREADS) k_pose(const PoseArgs a) {
    __shared__ int wcount[DEM_POSE_THREADS / 32], s_prefix;
    if (a.skip && *a.skip) return;  // the work-list count stays 0: the search kernel behind finds no tile
    const unsigned full = 0xffffffffu;
    const int p = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    bool valid = false;
    double d[3] = {0.0, 0.0, 0.0};
    d4 qi, qj;
    qi.x = qj.x = 1.0; qi.y = qi.z = qi.w = qj.y = qj.z = qj.w = 0.0;
    int2 ij = make_int2(0, 0);
    if (p < a.npairs) {
        ij = a.pairs[p];
        const d4 xi = load4d(static_cast<const PosT*>(a.pos), ij.x), xj = load4d(static_cast<const PosT*>(a.pos), ij.y);
        qi = load4d(static_cast<const PosT*>(a.quat), ij.x);
        qj = load4d(static_cast<const PosT*>(a.quat), ij.y);
        // minimum image (any nearest image serves here: the bit-exact predicate R13 belongs to the neighbour list)
        d[0] = xj.x - xi.x; d[1] = xj.y - xi.y; d[2] = DIM == 3 ? xj.z - xi.z : 0.0;
        d[0] -= a.box.L[0] * rint(d[0] * a.box.invL[0]);
        d[1] -= a.box.L[1] * rint(d[1] * a.box.invL[1]);
        if (DIM == 3) d[2] -= a.box.L[2] * rint(d[2] * a.box.invL[2]);
        valid = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < a.reach2;
    }
    // Compaction.  Inside a block the pairs keep their order; a block's slice of the work list is padded to a multiple of
    // 32 entries (pidx = -1) and placed with one atomicAdd, so every warp of the search kernel gets 32 consecutive
    // entries of ONE block: which pairs share a warp, and with it every sum downstream, is the same from run to run
    // although the order of the blocks' slices is not.
    const unsigned m = __ballot_sync(full, valid);
    if (lane == 0) wcount[warp] = __popc(m);
    __syncthreads();
    int tot = 0;
#pragma unroll
    for (int k = 0; k < DEM_POSE_THREADS / 32; ++k) tot += wcount[k];
    const int tot_pad = (tot + a.pad - 1) & ~(a.pad - 1);
    if (threadIdx.x == 0) {
        s_prefix = tot_pad ? atomicAdd(a.count, tot_pad) : 0;
        if (tot && a.counters) atomicAdd(a.counters, (unsigned long long)tot);
    }
    float Mi[9], R[9], t[3];
    if (valid) {
        const double qa[4] = {qi.x, qi.y, qi.z, qi.w}, qb[4] = {qj.x, qj.y, qj.z, qj.w};
        pair_pose<float>(qa, qb, d, Mi, R, t);
    } else if (p < a.npairs) {  // beyond the reach: contributes nothing, no record is written
        for (int sl = 0; sl < a.slices; ++sl) a.rflag[(size_t)p * a.slices + sl] = 0;
    }
    __syncthreads();
    if ((int)threadIdx.x < tot_pad - tot) a.pidx[s_prefix + tot + threadIdx.x] = make_int4(-1, 0, 0, 0);
    if (valid) {
        int wb = s_prefix;
        for (int k = 0; k < warp; ++k) wb += wcount[k];
        const int c = wb + __popc(m & ((1u << lane) - 1u));
        const size_t n = a.plane;
        DEM_ASSERT(c >= 0 && (size_t)c < n && s_prefix + tot_pad <= (int)n);
        f4 v;
        v.x = R[0]; v.y = R[1]; v.z = R[2]; v.w = R[3]; a.pose[c] = v;
        v.x = R[4]; v.y = R[5]; v.z = R[6]; v.w = R[7]; a.pose[n + c] = v;
        v.x = R[8]; v.y = t[0]; v.z = t[1]; v.w = t[2]; a.pose[2 * n + c] = v;
        a.pidx[c] = make_int4(p, ij.x, ij.y, 0);
    }
}

// ---- a3 with exact per-feature culling (3D, the library default) ----------------------------------------------------------
// k_pose plus the cull tests of k_pair_cull, done here because this kernel has the pose in registers and idle issue slots
// (it is bound by the latency of its gathers), while the search kernel behind it runs at 10 warps per SM: every feature
// of a particle lies within its circumradius R of its centre, so an outer feature of the other particle at R + rc_search or
// more from that centre cannot be a candidate against any of its features.  Per pair three bit masks come out (edges of
// j near i, vertices of j near i, vertices of i near j; at most DEM_CM_WORDS words), and only pairs with a surviving
// feature enter the work list at all.
#define DEM_CM_WORDS 8
template <typename PosT> __global__ void __launch_bounds__(DEM_POSE_THREADS) k_pose_cull(const PoseArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int wcount[DEM_POSE_THREADS / 32], s_prefix;
    if (a.skip && *a.skip) return;  // the work-list count stays 0: the search kernel behind finds no tile
    f4* sm = reinterpret_cast<f4*>(smem_raw);
    const bool same = a.sa.off == a.sb.off;
    for (int k = threadIdx.x; k < a.sa.len; k += blockDim.x) sm[k] = a.table[a.sa.off + k];
    if (!same)
        for (int k = threadIdx.x; k < a.sb.len; k += blockDim.x) sm[a.sa.len + k] = a.table[a.sb.off + k];
    const f4* AV = sm;
    const f4* BV = same ? sm : sm + a.sa.len;
    const f4* BOE = BV + a.sb.nv + 2 * a.sb.ne + 4 * a.sb.nf + 2 * a.sb.nfe;
    const unsigned full = 0xffffffffu;
    const int p = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    bool valid = false;
    double d[3] = {0.0, 0.0, 0.0};
    d4 qi, qj;
    qi.x = qj.x = 1.0; qi.y = qi.z = qi.w = qj.y = qj.z = qj.w = 0.0;
    int2 ij = make_int2(0, 0);
    if (p < a.npairs) {
        ij = a.pairs[p];
        const d4 xi = load4d(static_cast<const PosT*>(a.pos), ij.x), xj = load4d(static_cast<const PosT*>(a.pos), ij.y);
        qi = load4d(static_cast<const PosT*>(a.quat), ij.x);
        qj = load4d(static_cast<const PosT*>(a.quat), ij.y);
        d[0] = xj.x - xi.x; d[1] = xj.y - xi.y; d[2] = xj.z - xi.z;
        d[0] -= a.box.L[0] * rint(d[0] * a.box.invL[0]);
        d[1] -= a.box.L[1] * rint(d[1] * a.box.invL[1]);
        d[2] -= a.box.L[2] * rint(d[2] * a.box.invL[2]);
        valid = d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < a.reach2;
    }
    __syncthreads();  // the staged tables
    float Mi[9], R[9], t[3];
    unsigned cm[DEM_CM_WORDS];
#pragma unroll
    for (int w = 0; w < DEM_CM_WORDS; ++w) cm[w] = 0u;
    unsigned anybit = 0u;
    if (valid) {
        const double qa[4] = {qi.x, qi.y, qi.z, qi.w}, qb[4] = {qj.x, qj.y, qj.z, qj.w};
        pair_pose<float>(qa, qb, d, Mi, R, t);
        // in j's frame the centre of i is -R^T t: |R v + t| = |v + R^T t|, no rotation of the features is needed
        float tp[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) tp[k] = R[k] * t[0] + R[3 + k] * t[1] + R[6 + k] * t[2];
#pragma unroll
        for (int w = 0; w < DEM_CM_WORDS; ++w) {
            unsigned m = 0u;
            if (w < a.mw_e) {  // edges of j: nearest point of the segment to the centre of i
                const int l0 = 32 * w, n = min(32, a.sb.ne - l0);
                for (int k = 0; k < n; ++k) {
                    const f4 a0 = BOE[2 * (l0 + k)], a1 = BOE[2 * (l0 + k) + 1];
                    const float qx = a0.x + tp[0], qy = a0.y + tp[1], qz = a0.z + tp[2];
                    const float s = fminf(fmaxf(-(qx * a1.x + qy * a1.y + qz * a1.z), 0.f), a0.w);
                    const float cx = qx + s * a1.x, cy = qy + s * a1.y, cz = qz + s * a1.z;
                    m |= (cx * cx + cy * cy + cz * cz < a.cull_a2 ? 1u : 0u) << k;
                }
            } else if (w < a.mw_e + a.mw_vj) {  // vertices of j near i
                const int o0 = 32 * (w - a.mw_e), n = min(32, a.sb.nv - o0);
                for (int k = 0; k < n; ++k) {
                    const f4 v = BV[o0 + k];
                    const float qx = v.x + tp[0], qy = v.y + tp[1], qz = v.z + tp[2];
                    m |= (qx * qx + qy * qy + qz * qz < a.cull_a2 ? 1u : 0u) << k;
                }
            } else if (w < a.mw_e + a.mw_vj + a.mw_vi) {  // vertices of i near j: |R^T (v - t)| = |v - t|
                const int o0 = 32 * (w - a.mw_e - a.mw_vj), n = min(32, a.sa.nv - o0);
                for (int k = 0; k < n; ++k) {
                    const f4 v = AV[o0 + k];
                    const float qx = v.x - t[0], qy = v.y - t[1], qz = v.z - t[2];
                    m |= (qx * qx + qy * qy + qz * qz < a.cull_b2 ? 1u : 0u) << k;
                }
            }
            cm[w] = m;
            anybit |= m;
        }
    }
    const bool keep = valid && anybit != 0u;
    if (p < a.npairs && !keep)  // beyond the reach, or no feature within reach of the other particle: contributes nothing
        for (int sl = 0; sl < a.slices; ++sl) a.rflag[(size_t)p * a.slices + sl] = 0;
    // compaction as in k_pose
    const unsigned m = __ballot_sync(full, keep);
    if (lane == 0) wcount[warp] = __popc(m);
    __syncthreads();
    int tot = 0;
#pragma unroll
    for (int k = 0; k < DEM_POSE_THREADS / 32; ++k) tot += wcount[k];
    const int tot_pad = (tot + a.pad - 1) & ~(a.pad - 1);
    if (threadIdx.x == 0) {
        s_prefix = tot_pad ? atomicAdd(a.count, tot_pad) : 0;
    }
    if (a.counters) {  // pairs inside the reach (dem_get_counters out[0]), whether or not a feature survives
        const unsigned mv = __ballot_sync(full, valid);
        if (lane == 0 && mv) atomicAdd(a.counters, (unsigned long long)__popc(mv));
    }
    __syncthreads();
    if ((int)threadIdx.x < tot_pad - tot) a.pidx[s_prefix + tot + threadIdx.x] = make_int4(-1, 0, 0, 0);
    if (keep) {
        int wb = s_prefix;
        for (int k = 0; k < warp; ++k) wb += wcount[k];
        const int c = wb + __popc(m & ((1u << lane) - 1u));
        const size_t n = a.plane;
        DEM_ASSERT(c >= 0 && (size_t)c < n && s_prefix + tot_pad <= (int)n);
        f4 v;
        v.x = R[0]; v.y = R[1]; v.z = R[2]; v.w = R[3]; a.pose[c] = v;
        v.x = R[4]; v.y = R[5]; v.z = R[6]; v.w = R[7]; a.pose[n + c] = v;
        v.x = R[8]; v.y = t[0]; v.z = t[1]; v.w = t[2]; a.pose[2 * n + c] = v;
        a.pidx[c] = make_int4(p, ij.x, ij.y, 0);
#pragma unroll
        for (int w = 0; w < DEM_CM_WORDS; ++w)
            if (w < a.mw_e + a.mw_vj + a.mw_vi) a.cmask[(size_t)w * n + c] = cm[w];
    }
}

// ---- the kernel ---------------------------------------------------------------------------------------------------------
// One warp = 32 consecutive (pair, slice) items of one pair class (same shapes, same loop bounds).  TE / TV = packed
// outer pairs per sweep for edges / vertices (2 TE outer edges, 2 TV outer vertices share every inner-feature load).
template <int DIM, int TE, int TV, int MINB>
__global__ void __launch_bounds__(128, MINB) k_pair_fast(const PairArgs<float> a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FastShared* fs = reinterpret_cast<FastShared*>(smem_raw);
    unsigned* queue = reinterpret_cast<unsigned*>(smem_raw + 256);  // 4 warps x DEM_QCAP
    float* sacc_all = reinterpret_cast<float*>(queue + 4 * DEM_QCAP);  // 4 warps x 7 x 32
    unsigned* scnt_all = reinterpret_cast<unsigned*>(sacc_all + 4 * 7 * 32);  // 4 warps x 4
    f4* stage_pose = reinterpret_cast<f4*>(scnt_all + 16);                 // 4 warps x [2][3][32] float4 (R, t)
    int4* stage_pidx = reinterpret_cast<int4*>(stage_pose + 4 * 2 * 3 * 32);  // 4 warps x [2][32] (pair, i, j, 0)
    f4* sm = reinterpret_cast<f4*>(stage_pidx + 4 * 2 * 32);
    static_assert(sizeof(FastShared) <= 256, "FastShared header");
    // stage the shape-feature tables of the class (a1) into shared memory
    const bool same = a.sa.off == a.sb.off;
    for (int k = threadIdx.x; k < a.sa.len; k += blockDim.x) sm[k] = a.table[a.sa.off + k];
    if (!same)
        for (int k = threadIdx.x; k < a.sb.len; k += blockDim.x) sm[a.sa.len + k] = a.table[a.sb.off + k];
    ShapeView<float> A, B;
    A.nv = a.sa.nv; A.ne = a.sa.ne; A.nf = a.sa.nf;
    A.V = sm; A.E = A.V + A.nv; A.F = A.E + 2 * A.ne; A.FE = A.F + 4 * A.nf; A.OE = A.FE + 2 * a.sa.nfe;
    A.EB = A.OE + 2 * A.ne; A.FB = A.EB + A.ne;
    B.nv = a.sb.nv; B.ne = a.sb.ne; B.nf = a.sb.nf;
    B.V = same ? sm : sm + a.sa.len; B.E = B.V + B.nv; B.F = B.E + 2 * B.ne; B.FE = B.F + 4 * B.nf;
    B.OE = B.FE + 2 * a.sb.nfe;
    B.EB = B.OE + 2 * B.ne; B.FB = B.EB + B.ne;
    if (threadIdx.x == 0) {
        fs->A = A;
        fs->B = B;
        fs->pc = a.pc;
    }
    if (threadIdx.x < 16) scnt_all[threadIdx.x] = 0u;
    __syncthreads();

    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpCtx w;
    w.fs = fs;
    w.q = queue + warp * DEM_QCAP;
    w.sacc = sacc_all + warp * 7 * 32;
    w.scnt = scnt_all + warp * 4;
    w.qn = 0;
    w.lane = lane;
    w.nown = 32;
    const float nrc2 = -a.rc2_search;
    const int count = *a.count;                // pairs inside the reach, compacted by k_pose
    const int np_pad = (count + 31) & ~31;     // slices are warp-uniform
    const int tps = np_pad >> 5;               // tiles per slice
    const int n_wtiles = tps * a.slices;       // (a work list holds far fewer than 2^31 / 32 tiles: 96 bytes per pair)
    const size_t plane = a.plane;
    unsigned n_ee = 0u, n_vf = 0u, n_vfe = 0u;
    auto slice_terms = [&](int ob, int oe, unsigned& e_, unsigned& v_, unsigned& ve_) {
        if (DIM == 3) {
            const int oE_ = B.ne, oV_ = B.ne + B.nv;
            const int r1 = max(min(oe, oE_) - ob, 0), r2 = max(min(oe, oV_) - max(ob, oE_), 0),
                      r3 = max(min(oe, oV_ + A.nv) - max(ob, oV_), 0);
            e_ = (unsigned)(r1 * A.ne);
            v_ = (unsigned)(r2 * A.nf + r3 * B.nf);
            ve_ = (unsigned)(r2 * a.sa.nfe + r3 * a.sb.nfe);
        } else {
            const int r1 = max(min(oe, B.nv) - ob, 0), r2 = max(min(oe, B.nv + A.nv) - max(ob, B.nv), 0);
            e_ = (unsigned)(r1 * A.ne + r2 * B.ne);  // 2D: vertex-edge terms
            v_ = ve_ = 0u;
        }
    };
    unsigned t_ee = 0u, t_vf = 0u, t_vfe = 0u;  // per pair of an unsliced class: the same for every tile
    if (a.slices == 1) slice_terms(0, a.n_outer, t_ee, t_vf, t_vfe);
    // Each warp takes every (gridDim.x * 4)-th tile (one tile per warp unless the class has more tiles than the grid
    // cap).  The pose records of a warp's next tile are copied global -> shared with cp.async while the current tile is
    // being swept; each lane copies and later reads only its own records.
    const int wt_stride = (int)gridDim.x * 4;
    f4* spose = stage_pose + warp * (2 * 3 * 32);   // [2][3][32]
    int4* spidx = stage_pidx + warp * (2 * 32);     // [2][32]
    // tile -> (slice, first entry of the work list): no division for unsliced classes
    auto locate = [&](int wt_, int& slice_, int& c0_) {
        slice_ = a.slices == 1 ? 0 : wt_ / tps;
        c0_ = (wt_ - slice_ * tps) * 32;
    };
    auto stage = [&](int buf, int wt_, int c0_) {
        if (wt_ < n_wtiles) {
            const int c_ = c0_ + lane;
            DEM_ASSERT(c_ >= 0 && (size_t)count <= plane);
            if (c_ < count) {
#pragma unroll
                for (int k = 0; k < 3; ++k)  // R and t (R_i and d: pose_tail)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(
                                     spose + (buf * 3 + k) * 32 + lane)), "l"(a.pose + k * plane + c_));
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(
                                 spidx + buf * 32 + lane)), "l"(a.pidx + c_));
            }
        }
        asm volatile("cp.async.commit_group;");
    };
    // With a tile counter (a.tile, zeroed per evaluation) the grid is one resident wave and every warp takes its next
    // tile from the counter, one tile ahead of the one it sweeps: no warp waits for the slowest warp of its block and
    // the tables are staged once per block.
    auto next_tile = [&](int wt_) -> int {
        if (!a.tile) return wt_ + wt_stride;
        int v = 0;
        if (lane == 0) v = atomicAdd(a.tile, 1);
        return __shfl_sync(full, v, 0);
    };
    int buf = 0;
    int wt = a.tile ? next_tile(0) : (int)blockIdx.x * 4 + warp, slice = 0, c0 = 0;
    if (wt < n_wtiles) locate(wt, slice, c0);
    stage(0, wt, c0);
    for (int wt_next, slice_next, c0_next; wt < n_wtiles; wt = wt_next, slice = slice_next, c0 = c0_next, buf ^= 1) {
        const int c = c0 + lane;
        const bool in_list = c < count;
        wt_next = next_tile(wt);
        slice_next = c0_next = 0;
        if (wt_next < n_wtiles) locate(wt_next, slice_next, c0_next);
        stage(buf ^ 1, wt_next, c0_next);
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncwarp();  // the cooperative evaluation reads other lanes' staged poses
        w.sp = spose + buf * 3 * 32;
        w.touched = 0u;
        const bool valid = in_list && spidx[buf * 32 + lane].x >= 0;  // the work list is padded to whole warps per k_pose block
        if (!__any_sync(full, valid)) continue;                    // a tile of padding only
        float R[9], t[3];
        if (valid) {
            const f4 p0 = spose[(buf * 3 + 0) * 32 + lane], p1 = spose[(buf * 3 + 1) * 32 + lane],
                     p2 = spose[(buf * 3 + 2) * 32 + lane];
            R[0] = p0.x; R[1] = p0.y; R[2] = p0.z; R[3] = p0.w; R[4] = p1.x; R[5] = p1.y; R[6] = p1.z; R[7] = p1.w;
            R[8] = p2.x; t[0] = p2.y; t[1] = p2.z; t[2] = p2.w;
        } else {  // lanes without work sweep a far-away dummy so that the warp stays converged
#pragma unroll
            for (int k = 0; k < 9; ++k) R[k] = (k % 4 == 0) ? 1.f : 0.f;
            t[0] = t[1] = 1.0e4f;
            t[2] = DIM == 3 ? 1.0e4f : 0.f;
        }
        {

#pragma unroll
            for (int k = 0; k < 7; ++k) w.sacc[k * 32 + lane] = 0.f;
            const int ob = a.slices == 1 ? 0 : slice * a.n_outer / a.slices;   // (n_outer <= 3 x 2^15: no overflow)
            const int oe = a.slices == 1 ? a.n_outer : (slice + 1) * a.n_outer / a.slices;
            if (valid) {  // terms this lane sweeps (for the flop count; the kernel sweeps every term of its pairs)
                if (a.slices != 1) slice_terms(ob, oe, t_ee, t_vf, t_vfe);
                n_ee += t_ee;
                n_vf += t_vf;
                n_vfe += t_vfe;
            }
            if (DIM == 3) {
                const int oE = B.ne, oV = B.ne + B.nv;
                // (1) first sum of Eq. 1: edges of j (outer, packed) against edges of i (inner)
                for (int l0 = ob, le = min(oe, oE); l0 < le; l0 += 2 * TE) {
                    for (int k0 = 0; k0 < A.ne; k0 += 32) {
                        u64 np2x[TE], np2y[TE], np2z[TE], d2x[TE], d2y[TE], d2z[TE], g[TE];
                        float Llo[TE], Lhi[TE];
#pragma unroll
                        for (int tau = 0; tau < TE; ++tau) {
                            const int la = min(l0 + 2 * tau, le - 1), lb = min(l0 + 2 * tau + 1, le - 1);
                            const f4 a0 = B.OE[2 * la], a1 = B.OE[2 * la + 1], b0 = B.OE[2 * lb], b1 = B.OE[2 * lb + 1];
                            float pa[3], pb[3];
                            vertex_to_i<float>(a0.x, a0.y, a0.z, R, t, pa);
                            vertex_to_i<float>(b0.x, b0.y, b0.z, R, t, pb);
                            np2x[tau] = pk(-pa[0], -pb[0]);
                            np2y[tau] = pk(-pa[1], -pb[1]);
                            np2z[tau] = pk(-pa[2], -pb[2]);
                            d2x[tau] = pk(R[0] * a1.x + R[1] * a1.y + R[2] * a1.z, R[0] * b1.x + R[1] * b1.y + R[2] * b1.z);
                            d2y[tau] = pk(R[3] * a1.x + R[4] * a1.y + R[5] * a1.z, R[3] * b1.x + R[4] * b1.y + R[5] * b1.z);
                            d2z[tau] = pk(R[6] * a1.x + R[7] * a1.y + R[8] * a1.z, R[6] * b1.x + R[7] * b1.y + R[8] * b1.z);
                            g[tau] = fma2(d2z[tau], np2z[tau], fma2(d2y[tau], np2y[tau], mul2(d2x[tau], np2x[tau])));
                            Llo[tau] = a0.w;
                            Lhi[tau] = b0.w;
                        }
                        const int k1 = min(k0 + 32, A.ne);
                        unsigned mask[TE];
#pragma unroll
                        for (int tau = 0; tau < TE; ++tau) mask[tau] = 0u;
                        for (int k = k0; k < k1; ++k) {
                            const f4 e0 = A.E[2 * k], e1 = A.E[2 * k + 1];
#pragma unroll
                            for (int tau = 0; tau < TE; ++tau)
                                mask[tau] = push_sign(mask[tau], ee_eval(e0, e1, np2x[tau], np2y[tau], np2z[tau], d2x[tau],
                                                                         d2y[tau], d2z[tau], g[tau], Llo[tau], Lhi[tau], nrc2));
                        }
                        unsigned any = 0u;
#pragma unroll
                        for (int tau = 0; tau < TE; ++tau) any |= mask[tau];
                        if (__any_sync(full, any != 0u)) push_and_drain<TE>(w, PH_EE, mask, k1 - k0, k0, l0, le);
                    }
                }
                // (2) third sum of Eq. 1: vertices of j (outer, packed, i's frame) against faces of i
                for (int o0 = max(ob, oE) - oE, on = min(oe, oV) - oE; o0 < on; o0 += 2 * TV) {
                    for (int f0 = 0; f0 < A.nf; f0 += 32) {
                        u64 px[TV], py[TV], pz[TV];
#pragma unroll
                        for (int tau = 0; tau < TV; ++tau) {
                            const f4 va = B.V[min(o0 + 2 * tau, on - 1)], vb = B.V[min(o0 + 2 * tau + 1, on - 1)];
                            float pa[3], pb[3];
                            vertex_to_i<float>(va.x, va.y, va.z, R, t, pa);
                            vertex_to_i<float>(vb.x, vb.y, vb.z, R, t, pb);
                            px[tau] = pk(pa[0], pb[0]);
                            py[tau] = pk(pa[1], pb[1]);
                            pz[tau] = pk(pa[2], pb[2]);
                        }
                        const int f1 = min(f0 + 32, A.nf);
                        unsigned mask[TV];
#pragma unroll
                        for (int tau = 0; tau < TV; ++tau) mask[tau] = 0u;
                        sweep_faces<TV>(A, a.sa, f0, f1, px, py, pz, nrc2, mask);
                        unsigned any = 0u;
#pragma unroll
                        for (int tau = 0; tau < TV; ++tau) any |= mask[tau];
                        if (__any_sync(full, any != 0u)) push_and_drain<TV>(w, PH_VF_OWN, mask, f1 - f0, f0, o0, on);
                    }
                }
                // (3) second sum of Eq. 1: vertices of i (outer, packed, j's frame) against faces of j
                for (int o0 = max(ob, oV) - oV, on = min(oe, oV + A.nv) - oV; o0 < on; o0 += 2 * TV) {
                    for (int f0 = 0; f0 < B.nf; f0 += 32) {
                        u64 px[TV], py[TV], pz[TV];
#pragma unroll
                        for (int tau = 0; tau < TV; ++tau) {
                            const f4 va = A.V[min(o0 + 2 * tau, on - 1)], vb = A.V[min(o0 + 2 * tau + 1, on - 1)];
                            float pa[3], pb[3];
                            vertex_to_j<float>(va.x, va.y, va.z, R, t, pa);
                            vertex_to_j<float>(vb.x, vb.y, vb.z, R, t, pb);
                            px[tau] = pk(pa[0], pb[0]);
                            py[tau] = pk(pa[1], pb[1]);
                            pz[tau] = pk(pa[2], pb[2]);
                        }
                        const int f1 = min(f0 + 32, B.nf);
                        unsigned mask[TV];
#pragma unroll
                        for (int tau = 0; tau < TV; ++tau) mask[tau] = 0u;
                        sweep_faces<TV>(B, a.sb, f0, f1, px, py, pz, nrc2, mask);
                        unsigned any = 0u;
#pragma unroll
                        for (int tau = 0; tau < TV; ++tau) any |= mask[tau];
                        if (__any_sync(full, any != 0u)) push_and_drain<TV>(w, PH_VF_OTHER, mask, f1 - f0, f0, o0, on);
                    }
                }
            } else {
                // Eq. 2: vertices of j against edges of i (i's frame), then vertices of i against edges of j (j's frame)
#pragma unroll
                for (int side = 0; side < 2; ++side) {
                    const ShapeView<float>& In = side == 0 ? A : B;    // owner of the inner edges
                    const ShapeView<float>& Out = side == 0 ? B : A;   // owner of the outer vertices
                    const int base = side == 0 ? 0 : B.nv;
                    for (int o0 = max(ob, base) - base, on = min(oe, base + Out.nv) - base; o0 < on; o0 += 2 * TV) {
                        for (int k0 = 0; k0 < In.ne; k0 += 32) {
                            u64 px[TV], py[TV];
#pragma unroll
                            for (int tau = 0; tau < TV; ++tau) {
                                const f4 va = Out.V[min(o0 + 2 * tau, on - 1)], vb = Out.V[min(o0 + 2 * tau + 1, on - 1)];
                                float pa[3], pb[3];
                                if (side == 0) {
                                    vertex_to_i<float>(va.x, va.y, 0.f, R, t, pa);
                                    vertex_to_i<float>(vb.x, vb.y, 0.f, R, t, pb);
                                } else {
                                    vertex_to_j<float>(va.x, va.y, 0.f, R, t, pa);
                                    vertex_to_j<float>(vb.x, vb.y, 0.f, R, t, pb);
                                }
                                px[tau] = pk(pa[0], pb[0]);
                                py[tau] = pk(pa[1], pb[1]);
                            }
                            const int k1 = min(k0 + 32, In.ne);
                            unsigned mask[TV];
#pragma unroll
                            for (int tau = 0; tau < TV; ++tau) mask[tau] = 0u;
                            for (int k = k0; k < k1; ++k) {
                                const f4 e0 = In.E[2 * k], e1 = In.E[2 * k + 1];
#pragma unroll
                                for (int tau = 0; tau < TV; ++tau) {
                                    u64 sd, exc;
                                    edge2_eval(e0, e1, px[tau], py[tau], sd, exc);
                                    float lo, hi;
                                    upk(fma2(exc, exc, fma2(sd, sd, bc(nrc2))), lo, hi);
                                    mask[tau] = push_sign(mask[tau], fminf(lo, hi));
                                }
                            }
                            unsigned any = 0u;
#pragma unroll
                            for (int tau = 0; tau < TV; ++tau) any |= mask[tau];
                            if (__any_sync(full, any != 0u))
                                push_and_drain<TV>(w, side == 0 ? PH_VE_OWN : PH_VE_OTHER, mask, k1 - k0, k0, o0, on);
                        }
                    }
                }
            }
            if (w.qn > 0) {
                w.touched |= drain_terms(w.fs, w.q, w.sacc, w.scnt, w.qn, w.qn, w.sp, w.nown);
                w.qn = 0;
            }
            if (valid) {
                // a pair none of whose terms is inside the cutoff contributes nothing: its record flag is cleared and
                // no record is written (the reduction skips it)
                const int4 pe = spidx[buf * 32 + lane];
                const int pi = pe.x;
                DEM_ASSERT(pi < a.npairs && slice < a.slices);
                const size_t ri = (size_t)pi * a.slices + slice;
                a.rflag[ri] = (unsigned char)(w.touched & 1u);
                if (w.touched & 1u) {
                    float F[3], T[3];
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        F[k] = w.sacc[k * 32 + lane];
                        T[k] = w.sacc[(3 + k) * 32 + lane];
                    }
                    float Mi[9], dl[3];
                    pose_tail(a.pos, a.quat, a.pos_double, a.box, make_int2(pe.y, pe.z), Mi, dl);
                    float out[10];
                    pair_finish<float>(Mi, t, F, T, w.sacc[6 * 32 + lane], out);
                    f4* rec = a.rec + DEM_REC * ri;
                    f4 r0, r1, r2;
                    r0.x = out[0]; r0.y = out[1]; r0.z = out[2]; r0.w = out[9];
                    r1.x = out[3]; r1.y = out[4]; r1.z = out[5]; r1.w = dl[0];
                    r2.x = dl[1]; r2.y = dl[2]; r2.z = r2.w = 0.f;
                    rec[0] = r0; rec[1] = r1; rec[2] = r2;
                }
            }
        }
    }
    // counters: one atomic per warp per counter, after the hot loop
    __syncwarp();
    const unsigned long long s_ee = __reduce_add_sync(full, n_ee), s_vf = __reduce_add_sync(full, n_vf),
                             s_vfe = __reduce_add_sync(full, n_vfe);
    // (dem_get_counters reports the counters of the last dem_compute: inside dem_step they are not kept, a.counters is
    // null and the kernel ends without a single global atomic; bench.py's swept totals are kept while its timing is on)
    if (lane == 0) {
        if (a.counters) {
            if (s_ee) atomicAdd(a.counters + 4, s_ee);
            if (s_vf) atomicAdd(a.counters + 5, s_vf);
            if (s_vfe) atomicAdd(a.counters + 6, s_vfe);
            if (w.scnt[0]) atomicAdd(a.counters + 1, (unsigned long long)w.scnt[0]);
            if (w.scnt[1]) atomicAdd(a.counters + 2, (unsigned long long)w.scnt[1]);
            if (w.scnt[2]) atomicAdd(a.counters + 3, (unsigned long long)w.scnt[2]);
        }
        if (a.cum) {
            if (s_ee) atomicAdd(a.cum + 0, s_ee);
            if (s_vf) atomicAdd(a.cum + 1, s_vf);
            if (s_vfe) atomicAdd(a.cum + 2, s_vfe);
        }
    }
}

// bytes of dynamic shared memory k_pair_fast needs in front of the staged tables
static inline size_t fast_smem_header() {
    return 256 + sizeof(unsigned) * 4 * DEM_QCAP + sizeof(float) * 4 * 7 * 32 + sizeof(unsigned) * 16 +
           sizeof(f4) * 4 * 2 * 3 * 32 + sizeof(int4) * 4 * 2 * 32;
}

// ---- the kernel with exact per-feature culling (3D) ----------------------------------------------------------------------
// Every feature of particle i lies inside the ball of radius R_i (its circumradius) around its centre, so an outer
// feature of j whose distance from that centre is at least R_i + rc_search cannot be a candidate against ANY feature
// of i: the whole inner sweep for it can be skipped, exactly (PAPER.md:129 names such shape-local culling as the next
// step).  The test costs ~15 instructions per outer feature and needs no rotation (|R v + t| = |v + R^T t|).
// Because lanes disagree on which of their outer features survive, the survivors of the 32 pairs of a tile are
// compacted into a warp-private list of (owner lane, outer feature) items, and the sweeps run over ITEMS, two per lane
// in the halves of the packed registers (the halves may belong to different pairs: inner features are shared by the
// whole class, poses come from the staged records).  Candidates and their evaluation are as in k_pair_fast.
#define DEM_IQCAP 1024  // 32 lanes x 32 outer features per round

struct CullCtx {
    unsigned* iq;    // item list of the warp
    int iqn;         // items queued (warp-uniform)
    unsigned swept_ee, swept_vf, swept_vfe;  // this lane's swept edge-edge terms, vertex-face terms, face-edge tests
};

__device__ __forceinline__ void load_pose(const f4* sp, int nown, int owner, float* R, float* t) {
    const f4 p0 = sp[owner], p1 = sp[nown + owner], p2 = sp[2 * nown + owner];
    R[0] = p0.x; R[1] = p0.y; R[2] = p0.z; R[3] = p0.w; R[4] = p1.x; R[5] = p1.y; R[6] = p1.z; R[7] = p1.w;
    R[8] = p2.x; t[0] = p2.y; t[1] = p2.z; t[2] = p2.w;
}

// sweep the queued items of one phase, 64 per pass (two per lane)
// TWOLEVEL (large shapes): an item is first tested against the bounding spheres of the inner features (edges: midpoint
// and half length; faces: centre and radius; one packed test of ~10 instructions per inner feature for the lane's two
// items), and only the inner features whose sphere comes within the candidate cutoff of the item's own bounding sphere
// get the nearest-point search -- lane by lane, since the survivors differ between lanes (shape-local
// culling).  Measured on config 5 (truncated icosahedra: 90 edges, 32 faces; fork-to-join time of the three classes,
// from the lattice / thermalised): one level 115 / 83 us; faces two-level 107.6 / 81.6 (the choice); edges too
// 104.3 / 86.8 -- an edge item's sphere still meets ~9 of the partner's edge spheres, the union over a lane's two items
// and the maximum over the warp's lanes make 21 searches per pass where the uniform sweep makes 90 cheaper ones.
template <int PHASE, bool TWOLEVEL = false>
__device__ __forceinline__ void sweep_items(WarpCtx& w, CullCtx& cc, const ShapeView<float>& A, const ShapeView<float>& B,
                                            const ShapeDev& sda, const ShapeDev& sdb, float nrc2) {
    const unsigned full = 0xffffffffu;
    __syncwarp();
    for (int base = 0; base < cc.iqn; base += 64) {
        const int ia = base + w.lane, ib = ia + 32;
        const bool ok_a = ia < cc.iqn, ok_b = ib < cc.iqn;
        const unsigned ea = ok_a ? cc.iq[ia] : 0u, eb = ok_b ? cc.iq[ib] : ea;
        const int wa = (int)(ea >> 16), oa = (int)(ea & 0xffffu), wb = (int)(eb >> 16), ob = (int)(eb & 0xffffu);
        DEM_ASSERT(wa >= 0 && wa < w.nown && wb >= 0 && wb < w.nown);
        DEM_ASSERT(PHASE == PH_EE ? (oa < B.ne && ob < B.ne)
                   : PHASE == PH_VF_OWN ? (oa < B.nv && ob < B.nv)
                   : PHASE == PH_VF_OTHER ? (oa < A.nv && ob < A.nv) : ((oa & 0x7fff) < A.nv && (ob & 0x7fff) < A.nv));
        float Ra[9], ta[3], Rb[9], tb[3];
        load_pose(w.sp, w.nown, wa, Ra, ta);
        load_pose(w.sp, w.nown, wb, Rb, tb);
        if (!ok_a) ta[0] = tb[0] = 1.0e4f;  // idle lane: a far-away dummy keeps the warp converged
        if (PHASE == PH_EE) {
            const f4 a0 = B.OE[2 * oa], a1 = B.OE[2 * oa + 1], b0 = B.OE[2 * ob], b1 = B.OE[2 * ob + 1];
            float pa[3], pb[3];
            vertex_to_i<float>(a0.x, a0.y, a0.z, Ra, ta, pa);
            vertex_to_i<float>(b0.x, b0.y, b0.z, Rb, tb, pb);
            const u64 np2x = pk(-pa[0], -pb[0]), np2y = pk(-pa[1], -pb[1]), np2z = pk(-pa[2], -pb[2]);
            const float dax = Ra[0] * a1.x + Ra[1] * a1.y + Ra[2] * a1.z, dbx = Rb[0] * b1.x + Rb[1] * b1.y + Rb[2] * b1.z;
            const float day = Ra[3] * a1.x + Ra[4] * a1.y + Ra[5] * a1.z, dby = Rb[3] * b1.x + Rb[4] * b1.y + Rb[5] * b1.z;
            const float daz = Ra[6] * a1.x + Ra[7] * a1.y + Ra[8] * a1.z, dbz = Rb[6] * b1.x + Rb[7] * b1.y + Rb[8] * b1.z;
            const u64 d2x = pk(dax, dbx), d2y = pk(day, dby), d2z = pk(daz, dbz);
            const u64 g = fma2(d2z, np2z, fma2(d2y, np2y, mul2(d2x, np2x)));
            if constexpr (TWOLEVEL) {
                const float rcs = sqrtf(-nrc2), hla = 0.5f * a0.w, hlb = 0.5f * b0.w;
                // minus the midpoints of the two outer edges; their radii with the candidate cutoff added
                const u64 nmx = pk(-(pa[0] + hla * dax), -(pb[0] + hlb * dbx)), nmy = pk(-(pa[1] + hla * day), -(pb[1] + hlb * dby)),
                          nmz = pk(-(pa[2] + hla * daz), -(pb[2] + hlb * dbz));
                const u64 rho = pk(hla + rcs, hlb + rcs);
                for (int k0 = 0; k0 < A.ne; k0 += 32) {
                    const int k1 = min(k0 + 32, A.ne);
                    unsigned ma = 0u, mb = 0u;
                    for (int k = k0; k < k1; ++k) {
                        const f4 eb = A.EB[k];
                        const u64 dx = add2(bc(eb.x), nmx), dy = add2(bc(eb.y), nmy), dz = add2(bc(eb.z), nmz);
                        const u64 lim = add2(bc(eb.w), rho);
                        float lo, hi;
                        upk(fma2(neg2(lim), lim, fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)))), lo, hi);
                        ma = push_sign(ma, lo);
                        mb = push_sign(mb, hi);
                    }
                    unsigned mu = ma | mb;  // inner edges that one of the lane's two items has to search
                    while (__any_sync(full, mu != 0u)) {
                        const bool have = mu != 0u;
                        const int bit = have ? 31 - __clz((int)mu) : 0;
                        const int k = have ? k0 + (k1 - k0 - 1 - bit) : k0;
                        mu &= ~(1u << bit);
                        const float v = ee_eval(A.E[2 * k], A.E[2 * k + 1], np2x, np2y, np2z, d2x, d2y, d2z, g, a0.w, b0.w, nrc2);
                        push_lane(w, PHASE, PHASE, have && v < 0.f, k, wa, oa, ok_a, wb, ob, ok_b);
                        if (have) cc.swept_ee += (unsigned)((ok_a ? 1 : 0) + (ok_b ? 1 : 0));
                    }
                }
            } else {
                for (int k0 = 0; k0 < A.ne; k0 += 32) {
                    const int k1 = min(k0 + 32, A.ne);
                    unsigned mask = 0u;
#pragma unroll 1
                    for (int k = k0; k < k1; ++k)
                        mask = push_sign(mask, ee_eval(A.E[2 * k], A.E[2 * k + 1], np2x, np2y, np2z, d2x, d2y, d2z, g, a0.w,
                                                       b0.w, nrc2));
                    if (__any_sync(full, mask != 0u)) push_one(w, PHASE, PHASE, mask, k1 - k0, k0, wa, oa, ok_a, wb, ob, ok_b);
                }
                cc.swept_ee += (unsigned)((ok_a ? 1 : 0) + (ok_b ? 1 : 0)) * (unsigned)A.ne;
            }
        } else {
            // vertex-face items.  PH_VF_BOTH (one-shape classes: the faces of i and of j are the same table): bit 15 of
            // an item says which sum it belongs to, so both sums share one pass
            const ShapeView<float>& In = PHASE == PH_VF_OTHER ? B : A;
            const ShapeView<float>& Out = PHASE == PH_VF_OTHER ? A : B;
            const ShapeDev& sd = PHASE == PH_VF_OTHER ? sdb : sda;
            const bool oth_a = PHASE == PH_VF_OTHER || (PHASE == PH_VF_BOTH && (oa & 0x8000)),
                       oth_b = PHASE == PH_VF_OTHER || (PHASE == PH_VF_BOTH && (ob & 0x8000));
            const int va_i = oa & 0x7fff, vb_i = ob & 0x7fff;
            const f4 va = Out.V[va_i], vb = Out.V[vb_i];
            float pa[3], pb[3];
            if (oth_a)
                vertex_to_j<float>(va.x, va.y, va.z, Ra, ta, pa);
            else
                vertex_to_i<float>(va.x, va.y, va.z, Ra, ta, pa);
            if (oth_b)
                vertex_to_j<float>(vb.x, vb.y, vb.z, Rb, tb, pb);
            else
                vertex_to_i<float>(vb.x, vb.y, vb.z, Rb, tb, pb);
            u64 px[1] = {pk(pa[0], pb[0])}, py[1] = {pk(pa[1], pb[1])}, pz[1] = {pk(pa[2], pb[2])};
            if constexpr (TWOLEVEL) {
                const float rcs = sqrtf(-nrc2);
                const u64 npx = neg2(px[0]), npy = neg2(py[0]), npz = neg2(pz[0]);
                for (int f0 = 0; f0 < In.nf; f0 += 32) {
                    const int f1 = min(f0 + 32, In.nf);
                    unsigned ma = 0u, mb = 0u;
                    for (int f = f0; f < f1; ++f) {
                        const f4 fb = In.FB[f];
                        const u64 dx = add2(bc(fb.x), npx), dy = add2(bc(fb.y), npy), dz = add2(bc(fb.z), npz);
                        const float l = fb.w + rcs;
                        float lo, hi;
                        upk(fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc(-l * l)))), lo, hi);
                        ma = push_sign(ma, lo);
                        mb = push_sign(mb, hi);
                    }
                    unsigned mu = ma | mb;
                    while (__any_sync(full, mu != 0u)) {
                        const bool have = mu != 0u;
                        const int bit = have ? 31 - __clz((int)mu) : 0;
                        const int f = have ? f0 + (f1 - f0 - 1 - bit) : f0;
                        mu &= ~(1u << bit);
                        const f4 f3 = In.F[4 * f + 3];
                        unsigned m1[1] = {0u};
                        face_eval_any<1>(In.F + 4 * f, In.FE + 2 * (int)f3.x, (int)f3.y, px, py, pz, nrc2, m1);
                        push_lane(w, oth_a ? PH_VF_OTHER : PH_VF_OWN, oth_b ? PH_VF_OTHER : PH_VF_OWN, have && (m1[0] & 1u), f,
                                  wa, va_i, ok_a, wb, vb_i, ok_b);
                        if (have) {
                            const unsigned n2 = (unsigned)((ok_a ? 1 : 0) + (ok_b ? 1 : 0));
                            cc.swept_vf += n2;
                            cc.swept_vfe += n2 * (unsigned)f3.y;
                        }
                    }
                }
            } else {
                for (int f0 = 0; f0 < In.nf; f0 += 32) {
                    const int f1 = min(f0 + 32, In.nf);
                    unsigned mask[1] = {0u};
                    sweep_faces<1>(In, sd, f0, f1, px, py, pz, nrc2, mask);
                    if (__any_sync(full, mask[0] != 0u))
                        push_one(w, oth_a ? PH_VF_OTHER : PH_VF_OWN, oth_b ? PH_VF_OTHER : PH_VF_OWN, mask[0], f1 - f0, f0, wa,
                                 va_i, ok_a, wb, vb_i, ok_b);
                }
                cc.swept_vf += (unsigned)((ok_a ? 1 : 0) + (ok_b ? 1 : 0)) * (unsigned)In.nf;
                cc.swept_vfe += (unsigned)((ok_a ? 1 : 0) + (ok_b ? 1 : 0)) * (unsigned)sd.nfe;
            }
        }
    }
    cc.iqn = 0;
}

// Appending the lanes' surviving outer features (bit k of mask <=> feature o0 + k survives) to the item list, lane by
// lane (exclusive prefix of the lanes' counts: the order is fixed by the data), takes two steps so that the caller can
// sweep the list first when the new items would not fit: count_items returns the warp's total and the lane's offset,
// write_items stores the lane's items.
__device__ __forceinline__ int count_items(const WarpCtx& w, unsigned mask, int& offset) {
    const unsigned full = 0xffffffffu;
    const int cnt = __popc(mask);
    int incl = cnt;
#pragma unroll
    for (int dlt = 1; dlt < 32; dlt <<= 1) {
        const int y = __shfl_up_sync(full, incl, dlt);
        if (w.lane >= dlt) incl += y;
    }
    offset = incl - cnt;
    return __shfl_sync(full, incl, 31);
}
__device__ __forceinline__ void write_items(CullCtx& cc, unsigned mask, int owner, int o0, unsigned flag, int offset,
                                            int total) {
    int pos = cc.iqn + offset;
    DEM_ASSERT(cc.iqn >= 0 && cc.iqn + total <= DEM_IQCAP && offset >= 0 && offset + __popc(mask) <= total);
    while (mask) {
        const int b = __ffs(mask) - 1;
        mask &= mask - 1u;
        cc.iq[pos++] = ((unsigned)owner << 16) | flag | (unsigned)(o0 + b);
    }
    cc.iqn += total;
}
// the list is swept when the next batch would overflow it and at the end of a phase: passes run as full as possible
#define DEM_EMIT(PH, MASK, OWNER, O0, FLAG)                                               \
    do {                                                                                  \
        int off_;                                                                         \
        const unsigned m_ = (MASK);                                                       \
        const int tot_ = count_items(w, m_, off_);                                        \
        if constexpr (!NOOVF)                                                             \
            if (cc.iqn + tot_ > DEM_IQCAP) sweep_items<PH>(w, cc, A, B, a.sa, a.sb, nrc2); \
        write_items(cc, m_, (OWNER), (O0), (FLAG), off_, tot_);                           \
    } while (0)

// SAME: both particles of the class have the same shape.  ONESITE: one sweep site per phase (small code, for large shape
// tables) instead of one behind every emit site (the two owner slots' emits interleave: faster for small shapes).
// NOOVF: every item of a tile's phase fits the list (64 pairs x outer features <= DEM_IQCAP), so that the emit sites
// need no sweep of their own: three sweep sites in all (the instruction cache holds them).
// PRE (variants with emit sites only): the survivor masks come from k_pose_cull (a.cmask) / are tested here -- one
// kernel per case, because each case has sweep sites of its own and the thermalised kernel waits for instruction
// fetches a third of the time when it carries both.
template <int MINB, bool SAME, bool ONESITE, bool NOOVF, bool PRE>
__global__ void __launch_bounds__(128, MINB) k_pair_cull(const PairArgs<float> a) {
    // a warp tile is 64 pairs (two per lane: owner slots lane and lane + 32), so that the item passes run fuller
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FastShared* fs = reinterpret_cast<FastShared*>(smem_raw);
    unsigned* queue = reinterpret_cast<unsigned*>(smem_raw + 256);        // 4 warps x DEM_QCAP
    float* sacc_all = reinterpret_cast<float*>(queue + 4 * DEM_QCAP);      // 4 warps x 7 x 64
    unsigned* scnt_all = reinterpret_cast<unsigned*>(sacc_all + 4 * 7 * 64);  // 4 warps x 4
    f4* stage_pose = reinterpret_cast<f4*>(scnt_all + 16);                 // 4 warps x [3][64] float4 (R, t)
    int4* stage_pidx = reinterpret_cast<int4*>(stage_pose + 4 * 3 * 64);    // 4 warps x [64] (pair, i, j, 0)
    unsigned* items = reinterpret_cast<unsigned*>(stage_pidx + 4 * 64);     // 4 warps x DEM_IQCAP
    f4* sm = reinterpret_cast<f4*>(items + 4 * DEM_IQCAP);
    const bool same = SAME;
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // The kernel starts with a chain of dependent global loads (work-list length, pose records, masks) beside the staging
    // of the tables: the length is asked for first.  (Fetching every warp's first tile before the length has arrived was
    // measured: 1 % faster, but it reads the whole capacity of the work list, 57 MB instead of 11 MB on config 4.)
    const int count = *a.count;  // a multiple of 64 (k_pose pads its block slices)
    const size_t plane = a.plane;
    f4* spose = stage_pose + warp * (3 * 64);
    int4* spidx = stage_pidx + warp * 64;
    unsigned pm_e[2] = {0u, 0u}, pm_vj[2] = {0u, 0u}, pm_vi[2] = {0u, 0u};
    auto stage_tile = [&](int cbase_) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int own = lane + 32 * h, c_ = cbase_ + own;
#pragma unroll
            for (int k = 0; k < 3; ++k)  // R and t (R_i and d: pose_tail)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(
                                 spose + k * 64 + own)), "l"(a.pose + k * plane + c_));
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(spidx + own)),
                         "l"(a.pidx + c_));
        }
        asm volatile("cp.async.commit_group;");
    };
    // small shapes (one mask word per feature kind): the masks of k_pose_cull are asked for while the pose records are
    // on their way, instead of one dependent load per emit site
    auto load_masks = [&](int cbase_) {
        if constexpr (PRE && NOOVF) {
            const unsigned* cm = a.cmask + cbase_ + lane;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (a.mw_e) pm_e[h] = __ldg(cm + 32 * h);
                if (a.mw_vj) pm_vj[h] = __ldg(cm + (size_t)a.mw_e * plane + 32 * h);
                if (a.mw_vi) pm_vi[h] = __ldg(cm + (size_t)(a.mw_e + a.mw_vj) * plane + 32 * h);
            }
        }
    };
    for (int k = threadIdx.x; k < a.sa.len; k += blockDim.x) sm[k] = a.table[a.sa.off + k];
    if (!same)
        for (int k = threadIdx.x; k < a.sb.len; k += blockDim.x) sm[a.sa.len + k] = a.table[a.sb.off + k];
    ShapeView<float> A, B;
    A.nv = a.sa.nv; A.ne = a.sa.ne; A.nf = a.sa.nf;
    A.V = sm; A.E = A.V + A.nv; A.F = A.E + 2 * A.ne; A.FE = A.F + 4 * A.nf; A.OE = A.FE + 2 * a.sa.nfe;
    A.EB = A.OE + 2 * A.ne; A.FB = A.EB + A.ne;
    B.nv = a.sb.nv; B.ne = a.sb.ne; B.nf = a.sb.nf;
    B.V = same ? sm : sm + a.sa.len; B.E = B.V + B.nv; B.F = B.E + 2 * B.ne; B.FE = B.F + 4 * B.nf;
    B.OE = B.FE + 2 * a.sb.nfe;
    B.EB = B.OE + 2 * B.ne; B.FB = B.EB + B.ne;
    if (threadIdx.x == 0) {
        fs->A = A;
        fs->B = B;
        fs->pc = a.pc;
    }
    if (threadIdx.x < 16) scnt_all[threadIdx.x] = 0u;
    __syncthreads();

    WarpCtx w;
    w.fs = fs;
    w.q = queue + warp * DEM_QCAP;
    w.sacc = sacc_all + warp * 7 * 64;
    w.scnt = scnt_all + warp * 4;
    w.qn = 0;
    w.lane = lane;
    w.nown = 64;
    CullCtx cc;
    cc.iq = items + warp * DEM_IQCAP;
    cc.iqn = 0;
    cc.swept_ee = cc.swept_vf = cc.swept_vfe = 0u;
    const float nrc2 = -a.rc2_search;
    const long long n_wtiles = (long long)(count >> 6) * a.slices;
    w.sp = spose;
    for (long long wt = (long long)blockIdx.x * 4 + warp; wt < n_wtiles; wt += (long long)gridDim.x * 4) {
        const int slice = (int)(wt / (count >> 6)), cbase = (int)(wt - (long long)slice * (count >> 6)) * 64;
        __syncwarp();  // the previous tile's readers of the staged poses are done
        stage_tile(cbase);
        load_masks(cbase);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
        bool valid[2];
        valid[0] = spidx[lane].x >= 0;  // the work list is padded to whole tiles per k_pose block (pidx = -1)
        valid[1] = spidx[lane + 32].x >= 0;
        if (!__any_sync(full, valid[0] || valid[1])) continue;
        w.touched = 0u;
#pragma unroll
        for (int k = 0; k < 7; ++k) w.sacc[k * 64 + lane] = w.sacc[k * 64 + lane + 32] = 0.f;
        const int ob = (int)((long long)slice * a.n_outer / a.slices);
        const int oe = (int)((long long)(slice + 1) * a.n_outer / a.slices);
        const int oE = B.ne, oV = B.ne + B.nv;
        // this lane's two poses: t and R^T t (in j's frame the centre of i is -R^T t)
        float tq[2][3], tp[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            float R[9];
            load_pose(w.sp, 64, lane + 32 * h, R, tq[h]);
#pragma unroll
            for (int k = 0; k < 3; ++k) tp[h][k] = R[k] * tq[h][0] + R[3 + k] * tq[h][1] + R[6 + k] * tq[h][2];
        }
        if constexpr (ONESITE) {
            // Large shape tables (truncated icosahedra: 7 mask words per pair, faces of two sizes).  Every phase is ONE loop
            // over its (mask word, owner slot) units with ONE sweep site -- the item list is swept when the next batch
            // would overflow it and once when the phase ends.  The sweeps are big unrolled bodies; with a copy behind every
            // emit site the kernel has 28 k instructions, and a third of its stall samples are instruction fetches.
            // Survivor masks come from k_pose_cull (a.cmask) or are tested here (sliced pairs, masks that do not fit).
            const bool pre = a.cmask != nullptr;
            const unsigned* cm = a.cmask + (pre ? cbase + lane : 0);
            auto edge_word = [&](int l0, int n, float px_, float py_, float pz_) -> unsigned {
                unsigned m = 0u;
                for (int k = 0; k < n; ++k) {
                    const f4 a0 = B.OE[2 * (l0 + k)], a1 = B.OE[2 * (l0 + k) + 1];
                    const float qx = a0.x + px_, qy = a0.y + py_, qz = a0.z + pz_;
                    const float s = fminf(fmaxf(-(qx * a1.x + qy * a1.y + qz * a1.z), 0.f), a0.w);
                    const float cx = qx + s * a1.x, cy = qy + s * a1.y, cz = qz + s * a1.z;
                    m |= (cx * cx + cy * cy + cz * cz < a.cull_a2 ? 1u : 0u) << k;
                }
                return m;
            };
            auto vert_word = [&](const f4* V, int o0, int n, float sx, float sy, float sz, float lim2) -> unsigned {
                unsigned m = 0u;  // |v + s|^2 < lim2
                for (int k = 0; k < n; ++k) {
                    const f4 v = V[o0 + k];
                    const float qx = v.x + sx, qy = v.y + sy, qz = v.z + sz;
                    m |= (qx * qx + qy * qy + qz * qz < lim2 ? 1u : 0u) << k;
                }
                return m;
            };
            const int e_lo = pre ? 0 : ob, e_hi = pre ? B.ne : min(oe, oE);
            const int vj_lo = pre ? 0 : max(ob, oE) - oE, vj_hi = pre ? B.nv : min(oe, oV) - oE;
            const int vi_lo = pre ? 0 : max(ob, oV) - oV, vi_hi = pre ? A.nv : min(oe, oV + A.nv) - oV;
            const int nw_e = (max(e_hi - e_lo, 0) + 31) >> 5, nw_vj = (max(vj_hi - vj_lo, 0) + 31) >> 5,
                      nw_vi = (max(vi_hi - vi_lo, 0) + 31) >> 5;
            // phase 0: edges of j; then the two vertex-face sums, sharing their passes in one-shape classes
            for (int u = 0; u <= 2 * nw_e; ++u) {
                const bool last = u == 2 * nw_e;
                const int h = u & 1, wd = u >> 1, l0 = e_lo + 32 * wd;
                unsigned m = 0u;
                if (!last && (h ? valid[1] : valid[0]))
                    m = pre ? __ldg(cm + (size_t)wd * plane + 32 * h)
                            : edge_word(l0, min(32, e_hi - l0), h ? tp[1][0] : tp[0][0], h ? tp[1][1] : tp[0][1], h ? tp[1][2] : tp[0][2]);
                int off_;
                const int tot_ = count_items(w, m, off_);
                if (last || cc.iqn + tot_ > DEM_IQCAP) sweep_items<PH_EE, false>(w, cc, A, B, a.sa, a.sb, nrc2);
                if (!last) write_items(cc, m, lane + 32 * h, l0, 0u, off_, tot_);
            }
            auto vf_mask = [&](bool other, int wd, int h) -> unsigned {
                if (!(h ? valid[1] : valid[0])) return 0u;
                if (!other) {
                    if (wd >= nw_vj) return 0u;
                    const int o0 = vj_lo + 32 * wd;
                    return pre ? __ldg(cm + (size_t)(a.mw_e + wd) * plane + 32 * h)
                               : vert_word(B.V, o0, min(32, vj_hi - o0), h ? tp[1][0] : tp[0][0], h ? tp[1][1] : tp[0][1],
                                           h ? tp[1][2] : tp[0][2], a.cull_a2);
                }
                if (wd >= nw_vi) return 0u;
                const int o0 = vi_lo + 32 * wd;
                return pre ? __ldg(cm + (size_t)(a.mw_e + a.mw_vj + wd) * plane + 32 * h)
                           : vert_word(A.V, o0, min(32, vi_hi - o0), -(h ? tq[1][0] : tq[0][0]), -(h ? tq[1][1] : tq[0][1]),
                                       -(h ? tq[1][2] : tq[0][2]), a.cull_b2);
            };
            if constexpr (SAME) {
                const int nw = max(nw_vj, nw_vi);
                for (int u = 0; u <= 4 * nw; ++u) {
                    const bool last = u == 4 * nw;
                    const int h = u & 1, wd = u >> 2;
                    const bool other = (u >> 1) & 1;
                    const unsigned m = last ? 0u : vf_mask(other, wd, h);
                    int off_;
                    const int tot_ = count_items(w, m, off_);
                    if (last || cc.iqn + tot_ > DEM_IQCAP) sweep_items<PH_VF_BOTH, true>(w, cc, A, B, a.sa, a.sb, nrc2);
                    if (!last) write_items(cc, m, lane + 32 * h, (other ? vi_lo : vj_lo) + 32 * wd, other ? 0x8000u : 0u, off_, tot_);
                }
            } else {
                for (int u = 0; u <= 2 * nw_vj; ++u) {
                    const bool last = u == 2 * nw_vj;
                    const int h = u & 1, wd = u >> 1;
                    const unsigned m = last ? 0u : vf_mask(false, wd, h);
                    int off_;
                    const int tot_ = count_items(w, m, off_);
                    if (last || cc.iqn + tot_ > DEM_IQCAP) sweep_items<PH_VF_OWN, true>(w, cc, A, B, a.sa, a.sb, nrc2);
                    if (!last) write_items(cc, m, lane + 32 * h, vj_lo + 32 * wd, 0u, off_, tot_);
                }
                for (int u = 0; u <= 2 * nw_vi; ++u) {
                    const bool last = u == 2 * nw_vi;
                    const int h = u & 1, wd = u >> 1;
                    const unsigned m = last ? 0u : vf_mask(true, wd, h);
                    int off_;
                    const int tot_ = count_items(w, m, off_);
                    if (last || cc.iqn + tot_ > DEM_IQCAP) sweep_items<PH_VF_OTHER, true>(w, cc, A, B, a.sa, a.sb, nrc2);
                    if (!last) write_items(cc, m, lane + 32 * h, vi_lo + 32 * wd, 0u, off_, tot_);
                }
            }
        } else
        if constexpr (PRE && NOOVF) {
            // masks preloaded above; every item of a phase fits the list
#pragma unroll
            for (int h = 0; h < 2; ++h) DEM_EMIT(PH_EE, valid[h] ? pm_e[h] : 0u, lane + 32 * h, 0, 0u);
            sweep_items<PH_EE>(w, cc, A, B, a.sa, a.sb, nrc2);
            if constexpr (SAME) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    DEM_EMIT(PH_VF_BOTH, valid[h] ? pm_vj[h] : 0u, lane + 32 * h, 0, 0u);
                    DEM_EMIT(PH_VF_BOTH, valid[h] ? pm_vi[h] : 0u, lane + 32 * h, 0, 0x8000u);
                }
                sweep_items<PH_VF_BOTH>(w, cc, A, B, a.sa, a.sb, nrc2);
            } else {
#pragma unroll
                for (int h = 0; h < 2; ++h) DEM_EMIT(PH_VF_OWN, valid[h] ? pm_vj[h] : 0u, lane + 32 * h, 0, 0u);
                sweep_items<PH_VF_OWN>(w, cc, A, B, a.sa, a.sb, nrc2);
#pragma unroll
                for (int h = 0; h < 2; ++h) DEM_EMIT(PH_VF_OTHER, valid[h] ? pm_vi[h] : 0u, lane + 32 * h, 0, 0u);
                sweep_items<PH_VF_OTHER>(w, cc, A, B, a.sa, a.sb, nrc2);
            }
        } else if constexpr (PRE) {
            // the cull tests were done by k_pose_cull: one mask word per 32 outer features (slices == 1 on this path)
            const unsigned* cm = a.cmask + cbase + lane;
            for (int wd = 0; wd < a.mw_e; ++wd) {
#pragma unroll
                for (int h = 0; h < 2; ++h)
                    DEM_EMIT(PH_EE, valid[h] ? __ldg(cm + (size_t)wd * plane + 32 * h) : 0u, lane + 32 * h, 32 * wd, 0u);
            }
            sweep_items<PH_EE>(w, cc, A, B, a.sa, a.sb, nrc2);
            if constexpr (SAME) {
                for (int wd = 0; wd < a.mw_vj; ++wd) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const unsigned m2 = valid[h] ? __ldg(cm + (size_t)(a.mw_e + wd) * plane + 32 * h) : 0u;
                        const unsigned m3 = valid[h] ? __ldg(cm + (size_t)(a.mw_e + a.mw_vj + wd) * plane + 32 * h) : 0u;
                        DEM_EMIT(PH_VF_BOTH, m2, lane + 32 * h, 32 * wd, 0u);
                        DEM_EMIT(PH_VF_BOTH, m3, lane + 32 * h, 32 * wd, 0x8000u);
                    }
                }
                sweep_items<PH_VF_BOTH>(w, cc, A, B, a.sa, a.sb, nrc2);
            } else {
                for (int wd = 0; wd < a.mw_vj; ++wd) {
#pragma unroll
                    for (int h = 0; h < 2; ++h)
                        DEM_EMIT(PH_VF_OWN, valid[h] ? __ldg(cm + (size_t)(a.mw_e + wd) * plane + 32 * h) : 0u, lane + 32 * h,
                                 32 * wd, 0u);
                }
                sweep_items<PH_VF_OWN>(w, cc, A, B, a.sa, a.sb, nrc2);
                for (int wd = 0; wd < a.mw_vi; ++wd) {
#pragma unroll
                    for (int h = 0; h < 2; ++h)
                        DEM_EMIT(PH_VF_OTHER, valid[h] ? __ldg(cm + (size_t)(a.mw_e + a.mw_vj + wd) * plane + 32 * h) : 0u,
                                 lane + 32 * h, 32 * wd, 0u);
                }
                sweep_items<PH_VF_OTHER>(w, cc, A, B, a.sa, a.sb, nrc2);
            }
        } else {
            // (1) edges of j whose distance from i's centre is below R_i + rc_search
            for (int l0 = ob, le = min(oe, oE); l0 < le; l0 += 32) {
                const int n = min(32, le - l0);
    #pragma unroll
                for (int h = 0; h < 2; ++h) {
                    unsigned mask = 0u;
                    for (int k = 0; k < n; ++k) {
                        const f4 a0 = B.OE[2 * (l0 + k)], a1 = B.OE[2 * (l0 + k) + 1];
                        const float qx = a0.x + tp[h][0], qy = a0.y + tp[h][1], qz = a0.z + tp[h][2];
                        const float s = fminf(fmaxf(-(qx * a1.x + qy * a1.y + qz * a1.z), 0.f), a0.w);
                        const float cx = qx + s * a1.x, cy = qy + s * a1.y, cz = qz + s * a1.z;
                        mask |= (cx * cx + cy * cy + cz * cz < a.cull_a2 ? 1u : 0u) << k;
                    }
                    DEM_EMIT(PH_EE, valid[h] ? mask : 0u, lane + 32 * h, l0, 0u);
                }
            }
            sweep_items<PH_EE>(w, cc, A, B, a.sa, a.sb, nrc2);
            // (2) vertices of j near i: |R v + t| = |v + R^T t|;  (3) vertices of i near j: |R^T (v - t)| = |v - t|
            const int o2 = max(ob, oE) - oE, n2 = min(oe, oV) - oE, o3 = max(ob, oV) - oV, n3 = min(oe, oV + A.nv) - oV;
            if constexpr (SAME) {  // one shape: both sums sweep the same face table, so their survivors share the passes
                for (int c0 = 0; c0 < A.nv; c0 += 32) {
    #pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        unsigned m2 = 0u, m3 = 0u;
                        for (int k = 0; k < 32; ++k) {
                            const int o = c0 + k;
                            if (o >= A.nv) break;
                            const f4 v = A.V[o];
                            const float qx = v.x + tp[h][0], qy = v.y + tp[h][1], qz = v.z + tp[h][2];
                            const float rx = v.x - tq[h][0], ry = v.y - tq[h][1], rz = v.z - tq[h][2];
                            m2 |= (o >= o2 && o < n2 && qx * qx + qy * qy + qz * qz < a.cull_a2 ? 1u : 0u) << k;
                            m3 |= (o >= o3 && o < n3 && rx * rx + ry * ry + rz * rz < a.cull_b2 ? 1u : 0u) << k;
                        }
                        DEM_EMIT(PH_VF_BOTH, valid[h] ? m2 : 0u, lane + 32 * h, c0, 0u);
                        DEM_EMIT(PH_VF_BOTH, valid[h] ? m3 : 0u, lane + 32 * h, c0, 0x8000u);
                    }
                }
                sweep_items<PH_VF_BOTH>(w, cc, A, B, a.sa, a.sb, nrc2);
            } else {
                for (int o0 = o2; o0 < n2; o0 += 32) {
                    const int n = min(32, n2 - o0);
    #pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        unsigned mask = 0u;
                        for (int k = 0; k < n; ++k) {
                            const f4 v = B.V[o0 + k];
                            const float qx = v.x + tp[h][0], qy = v.y + tp[h][1], qz = v.z + tp[h][2];
                            mask |= (qx * qx + qy * qy + qz * qz < a.cull_a2 ? 1u : 0u) << k;
                        }
                        DEM_EMIT(PH_VF_OWN, valid[h] ? mask : 0u, lane + 32 * h, o0, 0u);
                    }
                }
                sweep_items<PH_VF_OWN>(w, cc, A, B, a.sa, a.sb, nrc2);
                for (int o0 = o3; o0 < n3; o0 += 32) {
                    const int n = min(32, n3 - o0);
    #pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        unsigned mask = 0u;
                        for (int k = 0; k < n; ++k) {
                            const f4 v = A.V[o0 + k];
                            const float qx = v.x - tq[h][0], qy = v.y - tq[h][1], qz = v.z - tq[h][2];
                            mask |= (qx * qx + qy * qy + qz * qz < a.cull_b2 ? 1u : 0u) << k;
                        }
                        DEM_EMIT(PH_VF_OTHER, valid[h] ? mask : 0u, lane + 32 * h, o0, 0u);
                    }
                }
                sweep_items<PH_VF_OTHER>(w, cc, A, B, a.sa, a.sb, nrc2);
            }
        }
        if (w.qn > 0) {
            w.touched |= drain_terms(w.fs, w.q, w.sacc, w.scnt, w.qn, w.qn, w.sp, w.nown);
            w.qn = 0;
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (!valid[h]) continue;
            const int own = lane + 32 * h;
            DEM_ASSERT(spidx[own].x < a.npairs && slice < a.slices);
            const size_t ri = (size_t)spidx[own].x * a.slices + slice;
            const bool hit = (w.touched >> h) & 1u;
            a.rflag[ri] = (unsigned char)hit;  // no contribution: no record is written, the reduction skips the pair
            if (!hit) continue;
            float F[3], T[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                F[k] = w.sacc[k * 64 + own];
                T[k] = w.sacc[(3 + k) * 64 + own];
            }
            float Mi[9], dl[3];
            pose_tail(a.pos, a.quat, a.pos_double, a.box, make_int2(spidx[own].y, spidx[own].z), Mi, dl);
            float out[10];
            pair_finish<float>(Mi, tq[h], F, T, w.sacc[6 * 64 + own], out);
            f4* rec = a.rec + DEM_REC * ri;
            f4 r0, r1, r2;
            r0.x = out[0]; r0.y = out[1]; r0.z = out[2]; r0.w = out[9];
            r1.x = out[3]; r1.y = out[4]; r1.z = out[5]; r1.w = dl[0];
            r2.x = dl[1]; r2.y = dl[2]; r2.z = r2.w = 0.f;
            rec[0] = r0; rec[1] = r1; rec[2] = r2;
        }
    }
    const unsigned s_ee = __reduce_add_sync(0xffffffffu, cc.swept_ee), s_vf = __reduce_add_sync(0xffffffffu, cc.swept_vf),
                   s_vfe = __reduce_add_sync(0xffffffffu, cc.swept_vfe);
    if (lane == 0) {  // inside dem_step a.counters is null: no global atomic at all (see k_pair_fast)
        if (a.counters) {
            if (w.scnt[0]) atomicAdd(a.counters + 1, (unsigned long long)w.scnt[0]);
            if (w.scnt[1]) atomicAdd(a.counters + 2, (unsigned long long)w.scnt[1]);
            if (w.scnt[2]) atomicAdd(a.counters + 3, (unsigned long long)w.scnt[2]);
            if (s_ee) atomicAdd(a.counters + 4, (unsigned long long)s_ee);
            if (s_vf) atomicAdd(a.counters + 5, (unsigned long long)s_vf);
            if (s_vfe) atomicAdd(a.counters + 6, (unsigned long long)s_vfe);
        }
        if (a.cum) {
            if (s_ee) atomicAdd(a.cum + 0, (unsigned long long)s_ee);
            if (s_vf) atomicAdd(a.cum + 1, (unsigned long long)s_vf);
            if (s_vfe) atomicAdd(a.cum + 2, (unsigned long long)s_vfe);
        }
    }
}

// bytes of dynamic shared memory k_pair_cull needs in front of the staged tables
static inline size_t cull_smem_header() {
    return 256 + sizeof(unsigned) * 4 * DEM_QCAP + sizeof(float) * 4 * 7 * 64 + sizeof(unsigned) * 16 +
           sizeof(f4) * 4 * 3 * 64 + sizeof(int4) * 4 * 64 + sizeof(unsigned) * 4 * DEM_IQCAP;
}

}  // namespace dem
