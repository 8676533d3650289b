// dt_propagate.cu -- kernel 1 (+2): propagate, light-time, project, footprint-cull, compact.
//
// Hot-path steps 1-7 of DESIGN.md (Algorithm 1 `SearchImages` + `FilterGPUIntersections`,
// PAPER.md:159-161, 168-169; the dense |images| x |orbits| result is NEVER materialised -- only the
// compacted hits leave the SM, cf. PAPER.md:202 where the paper stores "tens of bytes for each
// pair").
//
// Mapping: one orbit per thread (32 orbits per warp, kTileOrbits = 128 per CTA, 4 CTAs per SM); the thread walks the unit's
// exposures in time order carrying its Kepler state, so consecutive solves are warm-started.
// Exposure records (128 B each) are staged group by group (32 exposures = 4 KB) into shared memory
// by 1-D TMA bulk copies (cp.async.bulk, SASS UBLKCP) on a two-slot mbarrier ring; every lane
// reads the same record (broadcast).  Hits are compacted per warp and group with warp ballots:
// at every exposure the hitting lanes append their pixel offsets, in lane order, to the warp's
// shared-memory stage (so the stage is exposure-major, then lane-ascending); at the end of the
// group one lane reserves the range with a single integer atomicAdd, the warp copies the stage
// out with coalesced stores, and the 32 per-orbit hit masks are written as one coalesced 128-B row.
#include "dt_common.cuh"
#include "dt_orbit.cuh"
#include "dt_tma.cuh"

namespace dt {

#ifndef DT_K1_MIN_CTAS
#define DT_K1_MIN_CTAS 4           // resident CTAs per SM kernel 1 is compiled for (register budget)
#endif
#ifndef DT_K1_GATE_CTAS
#define DT_K1_GATE_CTAS 5          // the gate variant: its hot loop is latency-bound, one more CTA per SM pays
#endif
constexpr int kMaxSubsteps = 6;    // wide sub-steps of one Kepler step before the cold solve is cheaper
constexpr double kGateEpsMax = 0.35;   // AU: a looser remainder bound in the warp switches the group's gate off (the test
                                       // still removes every pair farther than ~eps / distance from the pointing)

struct __align__(128) PropSmem {
    ExpRec rec[2][kGroup];                       // 8 KB: two-slot ring of exposure groups
    uint32_t stage[kWarpsPerCta][kGroup * 32];   // 4 KB per warp: [warp][hit] staged pixel offsets
    double el[kTileOrbits * 6];                  // 48 B per orbit: the tile's elements (one bulk copy)
    float geph[11][kTileOrbits];                 // 44 B per orbit: the gate's group ephemeris (GroupEph), lane-contiguous
    float4 gexp[kWarpsPerCta][kGroup][2];        // 1 KB per warp: the group's exposures as the gate reads them, FP32:
                                                 // (t - tm, Rx, Ry, Rz), (tx, ty, tz, -)
    uint64_t full[2];
    uint64_t el_bar;
};

template <int MODE>
__global__ void __launch_bounds__(kTileOrbits, (MODE & kModeGate) ? DT_K1_GATE_CTAS : DT_K1_MIN_CTAS)
    k_propagate(const PropagateParams p)
{
    constexpr bool WARM = (MODE & kModeWarm) != 0;
    constexpr bool PRECULL = (MODE & kModePrecull) != 0;
    constexpr bool DENSE = (MODE & kModeDense) != 0;
    constexpr bool GATE = (MODE & kModeGate) != 0 && WARM && PRECULL;
    // both variants of a unit are enqueued; the one the policy does not name has nothing to do
    if (p.policy && (p.policy->select != 0) != GATE) return;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    PropSmem &sm = *reinterpret_cast<PropSmem *>(smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t orbit = (int64_t)blockIdx.x * kTileOrbits + tid;
    const int n_groups = (p.n_exp + kGroup - 1) / kGroup;
    const int g_begin = blockIdx.y * p.groups_per_split;
    const int g_end = min(n_groups, g_begin + p.groups_per_split);

    if (tid == 0) {
        mbar_init(&sm.full[0], 1);
        mbar_init(&sm.full[1], 1);
        mbar_init(&sm.el_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](int g) {   // thread 0 only
        const int slot = (g - g_begin) & 1;
        const int nrec = min(kGroup, p.n_exp - g * kGroup);
        const uint32_t bytes = (uint32_t)nrec * (uint32_t)sizeof(ExpRec);
        mbar_expect_tx(&sm.full[slot], bytes);
        bulk_g2s(&sm.rec[slot][0], p.exp + (size_t)g * kGroup, bytes, &sm.full[slot]);
    };
    if (tid == 0) {
        if (g_begin < g_end) issue(g_begin);
        if (g_begin + 1 < g_end) issue(g_begin + 1);
    }

    // ---- the tile's elements: ONE bulk copy into shared memory.  The source may be device memory or
    // page-locked HOST memory (dt_stack with DT_MEM_PINNED elements): the copy engine then reads the
    // tile over PCIe in one request while earlier CTAs compute, so no separate host->device copy of
    // the elements precedes the kernel; the first pass also leaves a device copy for later passes ----
    const int64_t tile_base = (int64_t)blockIdx.x * kTileOrbits;
    const int n_tile = (int)min((int64_t)kTileOrbits, p.n_orbits - tile_base);
    if (tid == 0) {
        const uint32_t bytes = (uint32_t)n_tile * 48u;
        mbar_expect_tx(&sm.el_bar, bytes);
        bulk_g2s(&sm.el[0], p.elements + tile_base * 6, bytes, &sm.el_bar);
    }
    mbar_wait(&sm.el_bar, 0);
    if (p.elements_copy && blockIdx.y == 0) {
        double2 *dst = reinterpret_cast<double2 *>(p.elements_copy + tile_base * 6);
        const double2 *src = reinterpret_cast<const double2 *>(&sm.el[0]);
        for (int k = tid; k < n_tile * 3; k += kTileOrbits) dst[k] = src[k];
    }

    // ---- per-orbit precompute (step 1) ----
    double el[6];
    const bool in_range = orbit < p.n_orbits;
#pragma unroll
    for (int k = 0; k < 6; ++k) el[k] = in_range ? sm.el[tid * 6 + k] : ((k == 0) ? -1.0 : 0.0);
    // epoch of M0: one per call, or one per orbit ("six orbital elements and an orbital epoch");
    // a non-finite epoch makes the orbit invalid
    const double t0 = p.t0_orbit ? (in_range ? p.t0_orbit[orbit] : 0.0) : p.t0;
    if (!isfinite(t0)) el[0] = -1.0;
    const Orbit o = orbit_setup(el, p.gm, p.cos_eps, p.sin_eps, p.inv_c, p.tan_fov);

    Kepler K;
    K.M = K.u = K.s = 0.0;
    K.c = 1.0;
    bool have_state = false;
    bool prev_refined = false;     // warp-uniform: the last exposure's pairs went through the refinement
    int since_sync = 0;            // warp-uniform: cull-quality steps since (sin E, cos E) were last exact
    unsigned long long n_refined = 0, n_cold = 0, n_hits = 0, n_sub = 0;
    unsigned int n_gated = 0;      // warp-uniform: exposures of this warp the group ephemeris gate removed

    for (int g = g_begin; g < g_end; ++g) {
        const int slot = (g - g_begin) & 1;
        const uint32_t parity = ((g - g_begin) >> 1) & 1;
        mbar_wait(&sm.full[slot], parity);
        const int nrec = min(kGroup, p.n_exp - g * kGroup);

        // (a warp that is culling needs no refresh: its chain is cull quality and self-correcting, and
        // the pairs that survive re-synchronise (sin E, cos E) exactly before they are refined)
        if (WARM && have_state && (!PRECULL || prev_refined)) {
            K = kepler_refresh(o.e, K);
            since_sync = 0;
        }

        bool gate_ready = false, gate_off = false;   // warp-uniform: this group's ephemeris exists / is of no use
        bool group_far = false;                      // warp-uniform: no lane can be near ANY exposure of the group
        uint32_t bits = 0;
        int cnt = 0;          // this lane's hits in the group
        int run = 0;          // the warp's hits in the group so far (warp-uniform)
        for (int jj = 0; jj < nrec; ++jj) {
            // ---- group ephemeris gate (dt_orbit.cuh, A25): ONE Taylor evaluation
            // per pair decides whether any lane can be near the exposure; a run of exposures none can be near costs
            // no Kepler step at all ----
            // (once the group's ephemeris exists also right after a refined exposure: in a survey that follows several
            // objects in turn, a warp's next exposure near its orbits is several exposures away; a warp that refines
            // every exposure of a group never pays for the ephemeris)
            if (GATE && !gate_off && (gate_ready || !prev_refined)) {
                if (!gate_ready) {
                    // lazily, once per group: mid-time and half-span
                    // of the group's exposures, in whatever order they come
                    // (any expansion time will do and the half-span only has to be an upper bound: FP32 offsets from
                    // the group's first record, reduced with two integer warp reductions on order-preserving keys)
                    const double t_first = sm.rec[slot][0].t;
                    const float off = __double2float_rn(sm.rec[slot][min(lane, nrec - 1)].t - t_first);
                    const uint32_t ob = __float_as_uint(off);
                    const uint32_t okey = ob ^ ((uint32_t)((int32_t)ob >> 31) | 0x80000000u);
                    const uint32_t klo = __reduce_min_sync(0xffffffffu, okey), khi = __reduce_max_sync(0xffffffffu, okey);
                    const float flo = __uint_as_float(klo ^ (((klo >> 31) - 1u) | 0x80000000u));
                    const float fhi = __uint_as_float(khi ^ (((khi >> 31) - 1u) | 0x80000000u));
                    const double tlo = t_first + (double)flo, thi = t_first + (double)fhi;
                    const double tm = 0.5 * (tlo + thi);
                    // + the rounding of the offsets (2^-24 relative each)
                    const double tau_max = fma(0.5 * (thi - tlo) + 1.2e-7 * fmax(fabs((double)flo), fabs((double)fhi)),
                                               1.000001, 1e-9);
                    const double a_orb = o.valid ? sm.el[tid * 6] : 1.0;
                    gate_ready = true;
                    // is the remainder bound of every lane tight enough to be of use?  Judged BEFORE the Kepler solve
                    // from the carried state: |r| over the group is no smaller than |r| there minus the longest way
                    // the object can go until the farthest exposure of the group (eccentric orbits next to a
                    // perihelion fail this; their warp then runs the group without the gate, at no cost)
                    if (have_state) {
                        const double t_cur = fma(K.M - o.M0, o.inv_n, t0);
                        const double far = fmax(fabs(thi - t_cur), fabs(tlo - t_cur));
                        const double rlow = fmax(a_orb * (1.0 - o.e), fma(-o.vmax, far, a_orb * fma(-o.e, K.c, 1.0)));
                        gate_off = !__all_sync(0xffffffffu,
                                               gate_eps_bound(p.gm, o.vmax, rlow, tau_max, p.tan_fov) < kGateEpsMax);
                    }
                    if (!gate_off) {
                        // lane j turns exposure j into what the test reads, FP32 (the warp's own copy: no CTA barrier)
                        float robs2 = 0.f;
                        if (lane < nrec) {
                            const ExpRec &y = sm.rec[slot][lane];
                            sm.gexp[warp][lane][0] = make_float4(__double2float_rn(y.t - tm), __double2float_rn(y.Rx),
                                                                 __double2float_rn(y.Ry), __double2float_rn(y.Rz));
                            sm.gexp[warp][lane][1] = make_float4(__double2float_rn(y.tx), __double2float_rn(y.ty),
                                                                 __double2float_rn(y.tz), 0.f);
                            robs2 = __double2float_ru(fma(y.Rx, y.Rx, fma(y.Ry, y.Ry, y.Rz * y.Rz)));
                        }
                        // max over the group (non-negative floats order like their bit patterns)
                        robs2 = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(robs2)));
                        const double r_obs_max = 1.000001 * sqrt((double)robs2);
                        // one polished Kepler solve at the mid-time (the carried state moves there: the chain stays at
                        // most half a group away from any exposure)
                        const double Mm = fma(o.n, tm - t0, o.M0);
                        Kepler Km = K;
                        bool okm = false;
                        if (have_state) Km = kepler_warm_wide<true>(o.e, K, Mm, okm);
                        if (!__all_sync(0xffffffffu, okm)) {
                            Km = kepler_cold(o.e, Mm);
                            n_cold += 1;
                        }
                        K = Km;
                        have_state = true;
                        since_sync = 0;
                        const GroupEph G = group_ephemeris(o, a_orb, K, tau_max, r_obs_max, p.gm, p.inv_c, p.tan_fov);
                        // the ephemeris lives in shared memory (lane-contiguous: conflict-free) and is read back at
                        // the head of every gated run, so that its registers are not live across the refinement
                        sm.geph[0][tid] = G.rx;
                        sm.geph[1][tid] = G.ry;
                        sm.geph[2][tid] = G.rz;
                        sm.geph[3][tid] = G.vx;
                        sm.geph[4][tid] = G.vy;
                        sm.geph[5][tid] = G.vz;
                        sm.geph[6][tid] = G.hx;
                        sm.geph[7][tid] = G.hy;
                        sm.geph[8][tid] = G.hz;
                        sm.geph[9][tid] = G.tq;
                        sm.geph[10][tid] = G.eps;
                        gate_off = !__all_sync(0xffffffffu, G.eps < (float)kGateEpsMax);
                        __syncwarp();
                        // one test for the whole group, where its pointings cluster (dt_orbit.cuh group_is_far)
                        if (p.group_bounds) {
                            const float4 b0 = p.group_bounds[3 * g], b1 = p.group_bounds[3 * g + 1],
                                         b2 = p.group_bounds[3 * g + 2];
                            group_far = __all_sync(0xffffffffu,
                                                   !o.valid || group_is_far(G.rx, G.ry, G.rz, __double2float_ru(o.vmax),
                                                                            __double2float_ru(tau_max),
                                                                            __double2float_ru(p.inv_c), b0, b1, b2));
                        }
                    }
                }
                if (group_far) {
                    if (DENSE && in_range) {              // dt_project: gated pairs are reported as culled
                        for (int q = jj; q < nrec; ++q) {
                            const int64_t k = (orbit * p.n_exp + (int64_t)g * kGroup + q) * 2;
                            if (p.radec) p.radec[k] = p.radec[k + 1] = nan("");
                            if (p.xy) p.xy[k] = p.xy[k + 1] = nan("");
                            if (p.pix) p.pix[k] = p.pix[k + 1] = -1;
                        }
                    }
                    n_gated += (unsigned)(nrec - jj);
                    break;
                }
                if (!gate_off) {
                    GroupEph G;
                    G.rx = sm.geph[0][tid];
                    G.ry = sm.geph[1][tid];
                    G.rz = sm.geph[2][tid];
                    G.vx = sm.geph[3][tid];
                    G.vy = sm.geph[4][tid];
                    G.vz = sm.geph[5][tid];
                    G.hx = sm.geph[6][tid];
                    G.hy = sm.geph[7][tid];
                    G.hz = sm.geph[8][tid];
                    G.tq = sm.geph[9][tid];
                    G.eps = sm.geph[10][tid];
                    const int j_first = jj;
                    // four exposures per step: independent dependency chains per lane, one loop overhead
                    bool stop = false;
                    while (!stop && jj < nrec) {
                        unsigned kept = 0;                 // bit q: some lane may be near exposure jj + q
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const int jq = min(jj + q, nrec - 1);
                            const float4 a = sm.gexp[warp][jq][0], b = sm.gexp[warp][jq][1];
                            const bool keep = !group_gate_culls(G, a.x, a.y, a.z, a.w, b.x, b.y, b.z);
                            kept |= (__ballot_sync(0xffffffffu, keep) != 0u ? 1u : 0u) << q;
                        }
                        const int valid = min(4, nrec - jj);
                        const int adv = min(kept ? __ffs(kept) - 1 : 4, valid);      // exposures gated by this step
                        stop = adv < valid;
                        if (DENSE && in_range) {          // dt_project: a gated pair is reported as culled
                            for (int q = 0; q < adv; ++q) {
                                const int64_t k = (orbit * p.n_exp + (int64_t)g * kGroup + jj + q) * 2;
                                if (p.radec) p.radec[k] = p.radec[k + 1] = nan("");
                                if (p.xy) p.xy[k] = p.xy[k + 1] = nan("");
                                if (p.pix) p.pix[k] = p.pix[k + 1] = -1;
                            }
                        }
                        jj += adv;
                    }
                    n_gated += (unsigned)(jj - j_first);
                    if (jj >= nrec) break;
                }
            }
            const ExpRec &x = sm.rec[slot][jj];
            const double dt = x.t - t0;
            const double M = fma(o.n, dt, o.M0);

            // ---- step 3: Kepler solve at t_j ----
            bool unpolished = false;       // warp-uniform: K still lacks its Newton polish
            if (WARM) {
                // order 3 when every lane's step is short (main-belt cadences), else order 4, else --
                // without spending the order-4 tail on a step that is outside its domain anyway --
                // the wide paths
                bool solved = false;
                unpolished = false;
                if (have_state) {
                    // the series is steered by the MUFU seed of 1/g in every mode (dt_orbit.cuh kepler_warm);
                    // the polished ORDER 4 step refines it first
                    WarmPre w = kepler_warm_pre(o.e, K, M, true);
                    if (__all_sync(0xffffffffu, kepler_warm_in_domain<3>(w))) {
                        // with the pre-cull the precision is deferred to the pairs that survive it
                        // (a warp whose last pair survived the cull -- a focused search -- polishes at
                        // once: deferring would cost it the geometric distance twice)
                        if (PRECULL && !prev_refined) {
                            // cull quality only: second-order series, no polish (<= 6e-6 rad in E, see
                            // orbit_setup for the cone slack that pays for it)
                            K = kepler_warm_finish<2, false>(o.e, K, M, w);
                            unpolished = true;
                            since_sync += 1;
                        } else {
                            K = kepler_warm_finish<3, true>(o.e, K, M, w);
                        }
                        solved = true;
                    } else if (__all_sync(0xffffffffu, kepler_warm_in_domain<4>(w))) {
                        if (PRECULL && !prev_refined) {
                            // cull quality on the order-4 domain: third-order series, no polish
                            // (<= 3.7e-6 rad in E over chained steps, inside the same 6e-6 budget)
                            K = kepler_warm_finish<3, false>(o.e, K, M, w);
                            unpolished = true;
                            since_sync += 1;
                        } else {
                            warm_refine_rg(w);
                            K = kepler_warm_finish<4>(o.e, K, M, w);
                        }
                        solved = true;
                    } else {
                        // some lane's step is too long (a long gap, or close to the perihelion of an
                        // eccentric orbit): one wide warm step from the same prefix, or equal wide
                        // sub-steps in M (count warp-uniform).  r <= 1 is the wide step's own domain;
                        // the margins leave room for the coefficients growing on the way to a
                        // perihelion (every step re-checks its domain)
                        const float r = __uint_as_float(
                            __reduce_max_sync(0xffffffffu, __float_as_uint(kepler_warm_need_pre(w))));
                        if (r < (float)kMaxSubsteps / 1.3f) {       // false for NaN
                            const int ns = (r <= 0.8f) ? 1 : (int)ceilf(1.3f * r);
                            Kepler Kc = K;
                            bool good = true;
                            const bool cullq = PRECULL && !prev_refined;   // second polish deferred to survivors
                            if (ns == 1) {
                                Kc = cullq ? kepler_warm_wide_finish<false>(o.e, K, M, w, good)
                                           : kepler_warm_wide_finish<true>(o.e, K, M, w, good);
                            } else {
                                const double M_from = K.M, dMs = (M - M_from) / (double)ns;
                                for (int sidx = 1; sidx <= ns; ++sidx) {
                                    bool oks;
                                    const double Ms = (sidx == ns) ? M : fma(dMs, (double)sidx, M_from);
                                    Kc = cullq ? kepler_warm_wide<false>(o.e, Kc, Ms, oks)
                                               : kepler_warm_wide<true>(o.e, Kc, Ms, oks);
                                    good = good && oks;
                                }
                            }
                            if (__all_sync(0xffffffffu, good)) {
                                K = Kc;
                                solved = true;
                                unpolished = cullq;
                                n_sub += 1;
                            }
                        }
                    }
                }
                if (!solved) {
                    K = kepler_cold(o.e, M);
                    n_cold += 1;
                }
                have_state = true;
            } else {
                K = kepler_cold(o.e, M);
                n_cold += 1;
            }

            // ---- step 4: geometric position and light-time ----
            const double X0 = K.c - o.e;
            const double dx0 = fma(o.Ax, X0, fma(o.Bx, K.s, -x.Rx));
            const double dy0 = fma(o.Ay, X0, fma(o.By, K.s, -x.Ry));
            const double dz0 = fma(o.Az, X0, fma(o.Bz, K.s, -x.Rz));
            const double rho2 = fma(dx0, dx0, fma(dy0, dy0, dz0 * dz0));

            bool near = true;
            if (PRECULL) {
                // conservative cone test on the GEOMETRIC direction (see orbit_setup)
                const double D0 = fma(dx0, x.tx, fma(dy0, x.ty, dz0 * x.tz));
                near = !(D0 * D0 < o.cos2_cull * rho2) && D0 > 0.0;
                // always refine close objects: there the error of the unpolished state could move the
                // direction by more than the cone's slack (and rho2 ~ 0 must not cull)
                near = near || !(rho2 > o.rho2_close);
            }
            bool hit = false;
            int32_t ix = -1, iy = -1;
            double xpix = 0.0, ypix = 0.0, qx = 0.0, qy = 0.0, qz = 0.0;
            const bool refine = !PRECULL || __any_sync(0xffffffffu, near);
            prev_refined = refine;
            if (refine) {
                n_refined += 1;
                double rho2r = rho2;
                if (unpolished) {
                    // the deferred polish, then the geometric distance again from the polished state
                    // (sin E, cos E) carry 1.6e-14 of truncation per cull-quality rotation: re-synchronise
                    // them exactly once more than a few such steps have piled up
                    // (<= 1e-13 in (sin E, cos E) after six steps = 1e-7 a / rho px), and at once when some lane of the
                    // warp is closer than a / 2 (a near-Earth pair: a / rho up to 20 would turn that into 2e-6 px)
                    const double a_orb = sm.el[tid * 6];
                    const bool close_pair = __any_sync(0xffffffffu, 4.0 * rho2 < a_orb * a_orb);
                    if (since_sync > 6 || (since_sync > 0 && close_pair)) {
                        K = kepler_resync(K);
                        since_sync = 0;
                    }
                    K = kepler_polish2(o.e, K);
                    const double X0p = K.c - o.e;
                    const double ax0 = fma(o.Ax, X0p, fma(o.Bx, K.s, -x.Rx));
                    const double ay0 = fma(o.Ay, X0p, fma(o.By, K.s, -x.Ry));
                    const double az0 = fma(o.Az, X0p, fma(o.Bz, K.s, -x.Rz));
                    rho2r = fma(ax0, ax0, fma(ay0, ay0, az0 * az0));
                }
                // one Goldschmidt step from the MUFU seed: 1.5e-12 relative, i.e. 3e-13 d of light-time
                const double rho0 = WARM ? sqrt_nr<1>(rho2r) : sqrt(rho2r);
                const double tau = rho0 * p.inv_c;
                const double M1 = fma(o.n, dt - tau, o.M0);
                Kepler K1;
                if (WARM) {
                    bool ok1;
                    K1 = kepler_warm<2>(o.e, K, M1, ok1);
                    if (!__all_sync(0xffffffffu, ok1)) K1 = kepler_newton_from(o.e, K, M1);
                } else {
                    K1 = kepler_newton_from(o.e, K, M1);
                }
                // ---- step 5: topocentric equatorial vector ----
                const double X1 = K1.c - o.e;
                qx = fma(o.Ax, X1, fma(o.Bx, K1.s, -x.Rx));
                qy = fma(o.Ay, X1, fma(o.By, K1.s, -x.Ry));
                qz = fma(o.Az, X1, fma(o.Bz, K1.s, -x.Rz));
                // ---- step 6: gnomonic projection (vector form) + pixelise ----
                const double D = fma(qx, x.tx, fma(qy, x.ty, qz * x.tz));
                // one Newton step from the MUFU seed: 1e-12 relative = 2e-9 px at the edge of a 4096-px footprint,
                // far inside the 1e-6 px guard band
                const double inv = WARM ? rcp_nr<1>(D) : 1.0 / D;
                const double xe = fma(qx, x.ex, fma(qy, x.ey, qz * x.ez));
                const double xn = fma(qx, x.nx, fma(qy, x.ny, qz * x.nz));
                xpix = fma(xe, inv, p.cx);
                ypix = fma(xn, inv, p.cy);
                const double xh = xpix + 0.5, yh = ypix + 0.5;
                // ---- step 7: footprint cull, in floating point before any integer conversion ----
                hit = o.valid && (D > 0.0) && (xh >= 0.0) && (xh < p.W) && (yh >= 0.0) && (yh < p.H);
                if (hit) {                               // 0 <= xh < W: truncation is the floor
                    ix = __double2int_rz(xh);
                    iy = __double2int_rz(yh);
                }
                if (!DENSE) {
                    // ---- cull + compaction, stage 1: ballot-compact this exposure's hits (only a warp that refined
                    // can have any) ----
                    const unsigned hm = __ballot_sync(0xffffffffu, hit);
                    if (hm) {
                        if (hit && DT_IN_BOUNDS(run + __popc(hm & ((1u << lane) - 1u)) < kGroup * 32 &&
                                                    (int64_t)iy * p.width + ix < (int64_t)p.W * (int64_t)p.H, p.counters + 7)) {
                            sm.stage[warp][run + __popc(hm & ((1u << lane) - 1u))] =
                                ((uint32_t)jj << kOffsetBits) | ((uint32_t)iy * (uint32_t)p.width + (uint32_t)ix);
                            bits |= 1u << jj;
                            cnt += 1;
                        }
                        run += __popc(hm);
                    }
                }
            }
            if (DENSE) {
                if (in_range) {
                    const int64_t k = (orbit * p.n_exp + (int64_t)g * kGroup + jj) * 2;
                    // with the pre-cull kept (dt_project under DT_FLAG_PROJECT_PRECULL) a pair whose warp the
                    // cull-quality cone test rejected is reported as culled: NaN, (-1, -1)
                    const bool rep = o.valid && refine;
                    if (p.radec) {
                        const double rho = sqrt(fma(qx, qx, fma(qy, qy, qz * qz)));
                        double ra = atan2(qy, qx);
                        if (ra < 0.0) ra += 2.0 * kPi;
                        p.radec[k] = rep ? ra : nan("");
                        p.radec[k + 1] = rep ? asin(qz / rho) : nan("");
                    }
                    if (p.xy) {
                        p.xy[k] = rep ? xpix : nan("");
                        p.xy[k + 1] = rep ? ypix : nan("");
                    }
                    if (p.pix) {
                        p.pix[k] = ix;
                        p.pix[k + 1] = iy;
                    }
                }
            }
        }

        n_hits += (unsigned long long)cnt;
        if (!DENSE) {
            // ---- stage 2: reserve the range, copy the stage out (exposure-major, coalesced) ----
            unsigned long long b0 = 0;
            if (run) {
                if (lane == 0) b0 = atomicAdd(p.counters, (unsigned long long)run);
                b0 = __shfl_sync(0xffffffffu, b0, 0);
                __syncwarp();
                uint32_t *dst = p.offsets + b0;
                if (DT_IN_BOUNDS((int64_t)b0 + run <= p.offsets_cap, p.counters + 7))
                    for (int k = lane; k < run; k += 32) dst[k] = sm.stage[warp][k];
            }
            const int64_t opad = (int64_t)blockIdx.x * kTileOrbits + tid;
            if (opad < p.n_pad) {
                p.mask[(int64_t)g * p.n_pad + opad] = bits;
                if (lane == 0) p.base[(int64_t)g * (p.n_pad >> 5) + (opad >> 5)] = b0;
            }
        }

        __syncthreads();   // every warp is done with rec[slot] (and its stage rows)
        if (tid == 0 && g + 2 < g_end) issue(g + 2);
    }

    // ---- statistics: one atomic per warp ----
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        n_refined += __shfl_xor_sync(0xffffffffu, n_refined, d);
        n_cold += __shfl_xor_sync(0xffffffffu, n_cold, d);
        n_hits += __shfl_xor_sync(0xffffffffu, n_hits, d);
        n_sub += __shfl_xor_sync(0xffffffffu, n_sub, d);
    }
    if (lane == 0 && p.counters) {
        atomicAdd(p.counters + 1, n_refined);
        atomicAdd(p.counters + 2, n_cold);
        if (n_hits) atomicAdd(p.counters + 3, n_hits);
        if (n_sub) atomicAdd(p.counters + 4, n_sub);
        if (GATE && n_gated) atomicAdd(p.counters + 6, 32ull * n_gated);   // pairs
    }
}

__global__ void k_group_bounds(const ExpRec *exp, int n_exp, double tan_fov, float4 *out);

template <int MODE>
static cudaError_t launch_mode(const PropagateParams &p, cudaStream_t stream)
{
    const size_t smem = sizeof(PropSmem);
    const int n_groups = (p.n_exp + kGroup - 1) / kGroup;
    const int splits = (n_groups + p.groups_per_split - 1) / p.groups_per_split;
    dim3 grid((unsigned)((p.n_orbits + kTileOrbits - 1) / kTileOrbits), (unsigned)splits);
    if ((MODE & kModeGate) && p.group_bounds)
        k_group_bounds<<<(unsigned)n_groups, 32, 0, stream>>>(p.exp, p.n_exp, p.tan_fov, p.group_bounds);
    k_propagate<MODE><<<grid, kTileOrbits, smem, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_propagate(const PropagateParams &p, int mode, cudaStream_t stream)
{
    if (p.n_orbits <= 0 || p.n_exp <= 0) return cudaSuccess;
    switch (mode) {
        case 0: return launch_mode<0>(p, stream);
        case 1: return launch_mode<1>(p, stream);
        case 2: return launch_mode<2>(p, stream);
        case 3: return launch_mode<3>(p, stream);
        case 4: return launch_mode<4>(p, stream);
        case 5: return launch_mode<5>(p, stream);
        case 6: return launch_mode<6>(p, stream);
        case 7: return launch_mode<7>(p, stream);
        case 11: return launch_mode<11>(p, stream);
        case 15: return launch_mode<15>(p, stream);
        default: return cudaErrorInvalidValue;
    }
}

// ---- per-group bounds of the gate's group-level test (dt_orbit.cuh group_is_far): one warp per exposure group ----
__global__ void __launch_bounds__(32) k_group_bounds(const ExpRec *exp, int n_exp, double tan_fov, float4 *out)
{
    const int g = blockIdx.x, lane = threadIdx.x;
    const int nrec = min(kGroup, n_exp - g * kGroup);
    const bool have = lane < nrec;
    const ExpRec x = exp[g * kGroup + min(lane, nrec - 1)];
    double sx = have ? x.tx : 0.0, sy = have ? x.ty : 0.0, sz = have ? x.tz : 0.0;
    double mx = have ? x.Rx : 0.0, my = have ? x.Ry : 0.0, mz = have ? x.Rz : 0.0;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        sx += __shfl_xor_sync(0xffffffffu, sx, d);
        sy += __shfl_xor_sync(0xffffffffu, sy, d);
        sz += __shfl_xor_sync(0xffffffffu, sz, d);
        mx += __shfl_xor_sync(0xffffffffu, mx, d);
        my += __shfl_xor_sync(0xffffffffu, my, d);
        mz += __shfl_xor_sync(0xffffffffu, mz, d);
    }
    const double sn = sqrt(fma(sx, sx, fma(sy, sy, sz * sz)));
    const bool axis = sn > 1e-3 * nrec;                       // pointings all around the sky: no axis
    const double cx = axis ? sx / sn : 1.0, cy = axis ? sy / sn : 0.0, cz = axis ? sz / sn : 0.0;
    mx /= nrec; my /= nrec; mz /= nrec;
    double cmin = have ? fma(x.tx, cx, fma(x.ty, cy, x.tz * cz)) : 1.0;                       // cos angle(t_j, c)
    const double ex = x.Rx - mx, ey = x.Ry - my, ez = x.Rz - mz;
    double dmax = have ? sqrt(fma(ex, ex, fma(ey, ey, ez * ez))) : 0.0;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        cmin = fmin(cmin, __shfl_xor_sync(0xffffffffu, cmin, d));
        dmax = fmax(dmax, __shfl_xor_sync(0xffffffffu, dmax, d));
    }
    if (lane == 0) {
        const double alpha = 1.01 * atan(tan_fov) + acos(fmin(fmax(cmin, -1.0), 1.0)) * 1.0001 + 1e-4;
        const bool ok = axis && alpha < 1.5 && isfinite(alpha) && isfinite(dmax);
        out[3 * g] = make_float4((float)cx, (float)cy, (float)cz, ok ? __double2float_rd(cos(alpha)) : -2.f);
        out[3 * g + 1] = make_float4((float)mx, (float)my, (float)mz, __double2float_ru(dmax * 1.0001 + 1e-6));
        out[3 * g + 2] = make_float4(ok ? __double2float_ru(sin(alpha)) : 1.f, 0.f, 0.f, 0.f);
    }
}

// ---- which kernel-1 variant the NEXT unit runs (GatePolicy, dt_k1.cuh): one thread, after every unit ----
// The gate pays where the warps cull (a blind search) and its remainder bounds are tight enough to gate; it costs
// where most pairs are refined anyway (a focused search: the variant without it is the faster binary there) or where
// the bounds are loose (eccentric near-Earth orbits).  Both are read off what the unit just did.
__global__ void k_gate_policy(GatePolicy *pol, const unsigned long long *counters, long long unit_pairs,
                              unsigned long long *max_unit_hits)
{
    if (max_unit_hits && counters[0] > *max_unit_hits) {
        *max_unit_hits = counters[0];
        __threadfence_system();
    }
    const unsigned long long refined = counters[1] - pol->refined0, gated = counters[6] - pol->gated0;
    pol->refined0 = counters[1];
    pol->gated0 = counters[6];
    int cooldown = pol->cooldown;
    const bool culling = (long long)refined * 4 < unit_pairs;
    if (pol->select != 0 && culling && (long long)gated * 4 < unit_pairs)
        cooldown = 64;                                   // the gate ran and gated little: off, tried again in 64 units
    else if (cooldown > 0)
        cooldown -= 1;
    pol->cooldown = cooldown;
    pol->select = (culling && cooldown == 0) ? 1 : 0;
}

cudaError_t launch_gate_policy(GatePolicy *policy, const unsigned long long *counters, int64_t unit_pairs,
                               unsigned long long *max_unit_hits, cudaStream_t stream)
{
    k_gate_policy<<<1, 1, 0, stream>>>(policy, counters, (long long)unit_pairs, max_unit_hits);
    return cudaGetLastError();
}

template <int MODE>
static cudaError_t set_smem_attr()
{
    return cudaFuncSetAttribute(k_propagate<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PropSmem));
}

// dynamic shared memory opt-in of every instantiation, for the CURRENT device (per device, not per process)
cudaError_t init_propagate_kernels()
{
    cudaError_t e;
    if ((e = set_smem_attr<0>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<1>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<2>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<3>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<4>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<5>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<6>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<7>()) != cudaSuccess) return e;
    if ((e = set_smem_attr<11>()) != cudaSuccess) return e;
    return set_smem_attr<15>();
}

}  // namespace dt
