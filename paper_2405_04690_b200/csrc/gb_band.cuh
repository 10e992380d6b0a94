// gb_band.cuh -- Algorithm 1 of the paper as a kernel.
// Included by gbfit.cu inside its anonymous namespace, after slow_part / fft_store / group_reduce.
//
// One CTA owns one band task j = (t, w, b) at a time: it stages the walker's residual r' and the noise weights
// 1/S_n of the task's bins [k_first, k_first + n_stage) (the paper's sub-bands b-1, b, b+1) in shared memory,
// then runs the task's proposals IN ORDER.  Each proposal is the SWAP evaluation of the batched path (two slow
// parts, two shared-memory FFTs, the five sums of Eq. 5) with the inner products read from the staged copy
// instead of global memory, the accept / reject decision beta dlnL + logq >= logu taken by thread 0 in FP64, and,
// when accepted, r' <- r' + h(theta_k) - h(theta'_k) in shared memory, theta_j[k] <- theta'_k in the caller's
// parameter array, and (write_back) the same window change added to the stored residual with FP64 atomics --
// the paper's "remove starting waveforms, add new group waveforms" of lines :608-613 done incrementally, so two
// bands of one walker that share a neighbour sub-band (b and b+2) never overwrite each other.
// Parallelism is across tasks only (the paper's design: the proposals of a band are a sequential chain).
#pragma once

struct BandArgs {
    const gb_band_task* tasks;
    int64_t n_tasks;
    double* params;
    const int32_t* prop_k;
    const double* prop_params;
    const double* prop_logq;
    const double* prop_logu;
    uint8_t* accepted_out;
    double* dlnL_out;
    const double* orbit;
    const cx* tw;
    double* resid;
    const double* psd;
    const int32_t* walker_psd;
    int64_t k_lo, n_f;
    int32_t n_walkers, n_psd, psd_is_inverse, max_stage;
    double Tobs, tau, Rmax;
    int64_t kmax;
    int32_t* errflag;
    cx* cache;               // [gridDim.x][kBandCacheSlots][2][N] windows of the current sources of each CTA's task
    // gb_band_sweep_generate: the proposal step runs inside the loop (gen != 0); prop_k / prop_params / prop_logq /
    // prop_logu are then OUTPUTS (what was generated for every proposal row)
    int32_t gen;
    gb_stretch st;           // seed, sweep, friends table (DEVICE), stretch scale, prior box, periodic flags
    int32_t* gen_k;
    double* gen_params;
    double* gen_logq;
    double* gen_logu;
};

// ---- the proposal step of Algorithm 1 (group stretch App. B :566-576; Eq. 14 :206-212) ----------
// Philox4x32-10 (Salmon et al. 2011): ten rounds of two 32x32 -> 64 multiplies and a key schedule by Weyl constants.
// Key = the 64-bit seed, counter = (proposal row, 0, block, sweep): the numbers of a proposal depend only on its row.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t* out) {
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0;  out[1] = c1;  out[2] = c2;  out[3] = c3;
}
// 52 random bits -> 0 < u < 1 (every step exact in FP64)
__device__ __forceinline__ double uniform52(uint32_t w0, uint32_t w1) {
    const double a = __dadd_rn(__dmul_rn((double)(w0 >> 6), 67108864.0), (double)(w1 >> 6));
    return __dmul_rn(__dadd_rn(a, 0.5), 1.0 / 4503599627370496.0);
}
__device__ __forceinline__ int32_t randint32(uint32_t w, int32_t n) { return (int32_t)__umulhi(w, (uint32_t)n); }

// First row s of the run of nf consecutive rows of the f0-sorted friends table that lie closest to f: the first s in
// [0, n_group - nf] at which trading row s for row s + nf would not bring the run closer,
//     P(s) = (f - g[s] > g[s + nf] - f)   is true below the answer and false from it on (g ascending),
// found by a 32-ary search of one warp (each lane probes one row per step).  [hlo, hhi] is a HINT where the answer
// probably lies (the friends of a band's sources sit next to each other): the first step probes both of its ends, and
// the search leaves the hint whenever P says so, so the result is that of the full search whatever the hint was.
// All 32 lanes of the warp must call it; all return the answer.
__device__ __forceinline__ int64_t friend_run_start(const double* __restrict__ group, int64_t n_group, int64_t nf, double f,
                                                    int lane, int64_t hlo, int64_t hhi) {
    const int64_t smax = n_group - nf;
    auto P = [&](int64_t p) { return (f - __ldg(group + 8 * p + 1)) > (__ldg(group + 8 * (p + nf) + 1) - f); };
    int64_t lo = 0, hi = smax;   // the answer lies in [lo, hi]
    if (hlo > 0 || hhi < smax) {
        const int64_t span = hhi - hlo;
        const int64_t p = hlo + (span * lane) / 31;                     // lane 0: hlo, lane 31: hhi
        const bool pred = p < smax ? P(p) : false;                      // (P(smax) counts as false: the answer is <= smax)
        const int c = __popc(__ballot_sync(0xffffffffu, pred));
        if (c == 0) hi = hlo;                                           // P(hlo) false: at or below the hint
        else if (c == 32) lo = hhi + 1;                                 // P(hhi) true: above the hint
        else {
            lo = hlo + (span * (c - 1)) / 31 + 1;
            hi = hlo + (span * c) / 31;
        }
    }
    while (hi > lo) {
        const int64_t span = hi - lo;
        const int64_t p = lo + (span * lane) / 32;                       // lo <= p < hi, non-decreasing in lane
        const int c = __popc(__ballot_sync(0xffffffffu, P(p)));         // lanes [0, c) are below the answer
        const int64_t nlo = c == 0 ? lo : lo + (span * (c - 1)) / 32 + 1;
        const int64_t nhi = c == 32 ? hi : lo + (span * c) / 32;
        lo = nlo;
        hi = nhi;
    }
    return lo;
}

// Current-source cache: a task with at most this many sources keeps the windows of its current sources in a per-CTA
// scratch area in global memory (8 KB per source for N = 256; all CTAs together ~150 MB, the live part ~40 MB, i.e.
// resident in the 126 MB L2).  A proposal then generates only the NEW waveform; the old one is copied in with
// cp.async while the new one is computed.  Same bits as regenerating it, 39 instead of 60 waveforms for a task of
// 9 sources and 30 proposals.
constexpr int kBandCacheSlots = 32;

template <int N>
constexpr size_t band_smem_bytes(int max_stage) {
    return (size_t)padded_len<N>() * sizeof(cx) * 4 + (size_t)max_stage * 48;
}

// resident CTAs per SM the register allocation aims at: what shared memory allows at the usual stage of 3 N bins
template <int N>
constexpr int band_min_blocks() { return N == 128 ? 6 : N == 256 ? 4 : N == 512 ? 2 : 1; }

// GEN: the proposal step runs inside the loop (gb_band_sweep_generate).  A template parameter rather than a flag: the loops
// of these kernels wait for instructions (ncu: 8-17 % of the warp samples), and each form is faster without the other's code.
template <int N, int GM, bool GEN>
__global__ void __launch_bounds__(Plan<N>::G * GM, band_min_blocks<N>()) gb_band_kernel(BandArgs a) {
    constexpr int PG = Plan<N>::G;   // FFT group: the first PG threads
    constexpr int G = PG * GM;       // threads of the CTA
    constexpr int S = N / G;
    constexpr int PN = padded_len<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx* bufA0 = reinterpret_cast<cx*>(smem_raw);      // old source theta_k
    cx* bufE0 = bufA0 + PN;
    cx* bufA1 = bufE0 + PN;                           // proposed source theta'_k
    cx* bufE1 = bufA1 + PN;
    cx* sRA = bufE1 + PN;                             // staged residual r' (A, E) and weights 1/S_n (A, E)
    cx* sRE = sRA + a.max_stage;
    double* sWA = reinterpret_cast<double*>(sRE + a.max_stage);
    double* sWE = sWA + a.max_stage;
    // records (step O1).  Window cache in use: the new source's record alternates between the two (step O1 runs one waveform
    // ahead) and the old source is known by its window start s_koff[k] alone; else 0 = the old source, 1 = the new one.
    // (Static shared memory is full: 4 CTAs of N = 256 with a stage of 768 bins fill the SM to the byte.)
    __shared__ __align__(16) SrcConst s_src[2];
    __shared__ double s_red[(G / 32) * 5 + 1];
    __shared__ int s_acc;
    __shared__ int s_gk[2], s_ginside[2];             // generated proposal (per record slot): k, inside the prior box
    __shared__ double s_glq[2], s_glu[2];             //                                       logq, logu
    __shared__ int32_t s_koff[kBandCacheSlots];       // window start of each cached current source, relative to t.k_first
    __shared__ double s_theta[kBandCacheSlots][8];    // generate mode: the band's CURRENT parameter rows ...
    __shared__ int64_t s_run[kBandCacheSlots];        // ... and where each one's run of friends starts in the table
    __shared__ int s_redo;                            // source whose run has to be searched again (it was just accepted)
    const int tid = threadIdx.x;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    cx* cache = a.cache ? a.cache + (size_t)blockIdx.x * kBandCacheSlots * 2 * N : nullptr;

    for (int64_t it = blockIdx.x; it < a.n_tasks; it += gridDim.x) {
        const gb_band_task t = a.tasks[it];
        const bool wb = (t.flags & GB_BAND_WRITE_BACK) != 0;
        const int wrow = (t.flags & GB_BAND_WRITE_OTHER) ? t.write_walker : t.walker;
        bool bad = t.walker < 0 || t.walker >= a.n_walkers || t.n_stage < 0 || t.n_stage > a.max_stage || t.n_src < 0 ||
                   (wb && (wrow < 0 || wrow >= a.n_walkers)) || (GEN && (t.n_src < 1 || t.n_stage < 1));
        int prow = 0;
        if (!bad) {
            prow = a.walker_psd ? a.walker_psd[t.walker] : (a.n_psd == 1 ? 0 : t.walker);
            bad = prow < 0 || prow >= a.n_psd;
        }
        if (bad) {
            if (tid == 0) atomicOr(a.errflag, 1);
            for (int p = tid; p < t.n_prop; p += G) {
                a.dlnL_out[t.prop_begin + p] = nan;
                a.accepted_out[t.prop_begin + p] = 0;
            }
            continue;
        }
        // ---- stage r' and the weights (zero weight marks a bin outside the stored band)
        const size_t nf = (size_t)a.n_f;
        const double* rA = a.resid + ((size_t)t.walker * 2 + 0) * nf * 2;   // staged from this row
        const double* rE = a.resid + ((size_t)t.walker * 2 + 1) * nf * 2;
        double* wA = a.resid + ((size_t)(wb ? wrow : t.walker) * 2 + 0) * nf * 2;   // accepted changes go to this row
        double* wE = a.resid + ((size_t)(wb ? wrow : t.walker) * 2 + 1) * nf * 2;
        const double* SA = a.psd + ((size_t)prow * 2 + 0) * nf;
        const double* SE = a.psd + ((size_t)prow * 2 + 1) * nf;
        const int64_t i_first = t.k_first - a.k_lo;   // stored element of staged bin 0
        for (int i = tid; i < t.n_stage; i += G) {
            const int64_t e = i_first + i;
            const bool ok = e >= 0 && e < a.n_f;
            cx ra = {0.0, 0.0}, re = {0.0, 0.0};
            double wa = 0.0, we = 0.0;
            if (ok) {
                const double2 a2 = __ldcg(reinterpret_cast<const double2*>(rA + 2 * e));
                const double2 e2 = __ldcg(reinterpret_cast<const double2*>(rE + 2 * e));
                ra = {a2.x, a2.y};
                re = {e2.x, e2.y};
                wa = a.psd_is_inverse ? SA[e] : 1.0 / SA[e];
                we = a.psd_is_inverse ? SE[e] : 1.0 / SE[e];
            }
            sRA[i] = ra;
            sRE[i] = re;
            sWA[i] = wa;
            sWE[i] = we;
        }
        cta_sync<G>();
        // ---- odd/even buffers: the staged row holds none of the band's own sources; subtract them
        const bool cached = cache != nullptr && t.n_src <= kBandCacheSlots;
        const bool subtract = (t.flags & GB_BAND_SUBTRACT_CURRENT) != 0;
        // Step O1 (one thread, ~1500 cycles) runs one waveform ahead wherever the next parameter row is known: while the
        // first PG threads transform a waveform, thread PG -- idle otherwise -- works out the record of the next one (the
        // band's next current source; with proposals given as inputs, the next proposal) into the other half of s_src.
        constexpr bool kAhead = GM > 1;
        int ns = 1;          // s_src slot of the next new-source record (toggles only with the window cache in use)
        bool have = false;   // s_src[ns] already holds it (uniform over the CTA)
        auto o1 = [&](const double* theta, SrcConst& dst) { seq_o1<N>(theta, a.Tobs, a.tau, a.Rmax, a.kmax, a.errflag, &dst); };
        // proposal p of the task can have its record made ahead: inputs-only form, window cache in use, k in range
        auto ahead_ok = [&](int p) -> bool {
            if (!kAhead || GEN || !cached || p >= t.n_prop) return false;
            const int kn = a.prop_k[(int64_t)t.prop_begin + p];
            return kn >= 0 && kn < t.n_src;
        };
        if (subtract || cached) {
            for (int sidx = 0; sidx < t.n_src; sidx++) {
                const double* theta = a.params + 8 * ((size_t)t.src_begin + sidx);
                if (!have) {
                    if (tid == 0) o1(theta, s_src[ns]);
                    cta_sync<G>();
                }
                const SrcConst* cur = &s_src[ns];
                const double* nxt = !kAhead || !cached ? nullptr : sidx + 1 < t.n_src ? theta + 8
                                              : ahead_ok(0) ? a.prop_params + 8 * (int64_t)t.prop_begin : nullptr;
                seq_window<N, G, PG>(cur, a.orbit, a.tw, bufA0, bufE0, a.Tobs, a.tau, tid);
                if (tid == PG && nxt) o1(nxt, s_src[ns ^ 1]);
                cta_sync<G>();
                const int64_t j0 = cur->kmin - t.k_first;
                if (cached && tid == 0) s_koff[sidx] = (int32_t)(cur->kmin - t.k_first);
#pragma unroll
                for (int m = 0; m < S; m++) {
                    const int j = tid + G * m;
                    const cx ha = bufA0[pad_idx<N>(j)], he = bufE0[pad_idx<N>(j)];
                    if (cached) {
                        cache[((size_t)sidx * 2 + 0) * N + j] = ha;
                        cache[((size_t)sidx * 2 + 1) * N + j] = he;
                    }
                    const int64_t i = j0 + j;
                    const int64_t e = i_first + i;
                    if (subtract && i >= 0 && i < t.n_stage && e >= 0 && e < a.n_f) {
                        sRA[i] = {sRA[i].re - ha.re, sRA[i].im - ha.im};
                        sRE[i] = {sRE[i].re - he.re, sRE[i].im - he.im};
                    }
                }
                cta_sync<G>();
                have = nxt != nullptr;
                if (cached) ns ^= 1;
            }
        }

        // ---- the proposals of the band, in order
        // friends search hint: the rows of the friends table inside the staged frequency range, widened by n_friends
        // (proposals are confined to the stage, so the run of a current source starts in there; the search checks it anyway)
        int64_t hint_lo = 0, hint_hi = 0;
        // bands of up to kBandCacheSlots sources keep their current parameter rows and the start of each source's run of
        // friends on chip: the search (4-5 dependent table probes) then leaves the per-proposal chain -- it is done once
        // per source here, all warps taking sources in turn, and again only for a source whose proposal was accepted
        const bool gen_cached = GEN && t.n_src <= kBandCacheSlots;
        if (GEN) {
            const int lane = tid & 31;
            const int64_t nfr = min((int64_t)a.st.n_friends, a.st.n_group);
            const double f_lo = (double)t.k_first / a.Tobs, f_hi = (double)(t.k_first + t.n_stage) / a.Tobs;
            hint_lo = max((int64_t)0, friend_run_start(a.st.group, a.st.n_group, 0, f_lo, lane, 0, a.st.n_group) - nfr);
            hint_hi = min(a.st.n_group - nfr, friend_run_start(a.st.group, a.st.n_group, 0, f_hi, lane, 0, a.st.n_group));
            if (hint_hi < hint_lo) hint_hi = hint_lo;
            if (gen_cached) {
                for (int i = tid; i < 8 * t.n_src; i += G) s_theta[i >> 3][i & 7] = a.params[8 * (size_t)t.src_begin + i];
                if (tid == 0) s_redo = -1;
                cta_sync<G>();
                for (int kk = tid >> 5; kk < t.n_src; kk += G / 32) {
                    const int64_t s0 = friend_run_start(a.st.group, a.st.n_group, nfr, s_theta[kk][1], lane, hint_lo, hint_hi);
                    if (lane == 0) s_run[kk] = s0;
                }
                cta_sync<G>();
            }
        }
        // "k <- randint(0, g_j); theta'_k <- Make Proposal on theta" of proposal row ipx by ONE warp (lane =
        // 0 .. 31), from the CURRENT theta_k: Philox block 0 -> k, the friend, z; block 1 -> the uniform of the accept step.
        // Lane c < 8 owns coordinate c of theta'; every product and sum is rounded on its own (the oracle is built without
        // FMA contraction), so k and theta' agree with it bit for bit.  Results: record slot `slot` of s_src / s_g*, and the
        // proposal's rows of the gen_* outputs.
        auto generate = [&](int64_t ipx, int slot, int lane) {
            uint32_t w0[4], w1[4];
            const uint32_t key0 = (uint32_t)(a.st.seed & 0xffffffffu), key1 = (uint32_t)(a.st.seed >> 32);
            philox4x32_10((uint32_t)ipx, 0u, 0u, a.st.sweep, key0, key1, w0);
            philox4x32_10((uint32_t)ipx, 0u, 1u, a.st.sweep, key0, key1, w1);
            const int kk = randint32(w0[0], t.n_src);
            const double* th = gen_cached ? s_theta[kk] : a.params + 8 * ((size_t)t.src_begin + kk);
            const int64_t nf = a.st.n_friends < a.st.n_group ? a.st.n_friends : a.st.n_group;
            const int32_t jf = randint32(w0[1], (int32_t)nf);
            if (gen_cached && s_redo >= 0) {   // the source accepted last has moved: its run of friends again
                const int kr = s_redo;
                const int64_t sr = friend_run_start(a.st.group, a.st.n_group, nf, s_theta[kr][1], lane, hint_lo, hint_hi);
                __syncwarp();
                if (lane == 0) {
                    s_run[kr] = sr;
                    s_redo = -1;
                }
                __syncwarp();
            }
            const int64_t s0 = gen_cached ? s_run[kk]
                                          : friend_run_start(a.st.group, a.st.n_group, nf, th[1], lane, hint_lo, hint_hi);
            const int64_t row = s0 + jf;
            const double ua = uniform52(w0[2], w0[3]);
            const double tz = __dadd_rn(__dmul_rn(__dadd_rn(a.st.stretch_a, -1.0), ua), 1.0);
            const double z = __ddiv_rn(__dmul_rn(tz, tz), a.st.stretch_a);    // g(z) ~ z^(-1/2) on [1/a, a]
            const int c = lane & 7;
            const double xa = __ldg(a.st.group + 8 * row + c);
            double x = __dadd_rn(xa, __dmul_rn(z, __dadd_rn(th[c], -xa)));      // Eq. 14
            const double lo = a.st.lo[c], hi = a.st.hi[c];
            if (a.st.periodic[c]) {
                const double period = __dadd_rn(hi, -lo);
                x = __dadd_rn(x, -__dmul_rn(period, floor(__ddiv_rn(__dadd_rn(x, -lo), period))));
            }
            const bool in_c = x >= lo && x <= hi;
            bool inside = (__ballot_sync(0xffffffffu, in_c) & 0xffu) == 0xffu;
            if (lane < 8) a.gen_params[8 * ipx + lane] = x;
            double pr[8];
#pragma unroll
            for (int cc = 0; cc < 8; cc++) pr[cc] = __shfl_sync(0xffffffffu, x, cc);
            {   // samples may go halfway into the neighbouring sub-bands: the window of theta' must
                // stay on the staged bins, else the prior is zero
                const int64_t kmin_p = (int64_t)floor(__dmul_rn(pr[1], a.Tobs) + 0.5) - N / 2;
                if (kmin_p < t.k_first || kmin_p + N > t.k_first + t.n_stage) inside = false;
            }
            if (lane == 0) {
                const double lq = 7.0 * log(z), lu = log(uniform52(w1[0], w1[1]));   // z^(D-1), D = 8
                a.gen_k[ipx] = kk;
                a.gen_logq[ipx] = lq;
                a.gen_logu[ipx] = lu;
                s_gk[slot] = kk;
                s_ginside[slot] = inside ? 1 : 0;
                s_glq[slot] = lq;
                s_glu[slot] = lu;
                if (!inside) {          // zero prior: rejected without a likelihood evaluation
                    a.dlnL_out[ipx] = nan;
                    a.accepted_out[ipx] = 0;
                }
            }
            if (lane == 1 && inside) o1(pr, s_src[slot]);   // step O1 of the proposed source, from registers
        };
        for (int p = 0; p < t.n_prop; p++) {
            const int64_t ip = (int64_t)t.prop_begin + p;
            int k;
            const double* theta_p;
            if (GEN) {
                if (tid < 32) generate(ip, ns, tid);
                cta_sync<G>();
                const bool inside = s_ginside[ns] != 0;
                k = s_gk[ns];
                if (!inside) {                  // uniform over the CTA
                    cta_sync<G>();              // slot ns is rewritten by the next proposal
                    have = false;
                    continue;
                }
                theta_p = a.gen_params + 8 * ip;
            } else {
                k = a.prop_k[ip];
                theta_p = a.prop_params + 8 * ip;
            }
            if (k < 0 || k >= t.n_src) {   // uniform over the CTA
                if (tid == 0) {
                    atomicOr(a.errflag, 1);
                    a.dlnL_out[ip] = nan;
                    a.accepted_out[ip] = 0;
                }
                continue;
            }
            double* theta_k = a.params + 8 * ((size_t)t.src_begin + k);
            const int nw = ns;   // slot of this proposal's record
            const bool nxt_ok = ahead_ok(p + 1);
            if (!have) {   // step O1 for the old (thread 0) and the proposed (thread 1) source, as far as they are still missing
                if (GEN ? (!cached && tid == 0) : (cached ? tid == 1 : tid < 2)) o1(tid == 0 ? theta_k : theta_p, s_src[tid == 0 ? 0 : nw]);
            }
            if (cached) {   // the old window comes from the cache while the new one is generated
#pragma unroll
                for (int m = 0; m < S; m++) {
                    const int j = tid + G * m;
                    cp_async16(&bufA0[pad_idx<N>(j)], &cache[((size_t)k * 2 + 0) * N + j]);
                    cp_async16(&bufE0[pad_idx<N>(j)], &cache[((size_t)k * 2 + 1) * N + j]);
                }
                cp_async_commit();
            }
            cta_sync<G>();
            if (!cached) {
                seq_window<N, G, PG>(&s_src[0], a.orbit, a.tw, bufA0, bufE0, a.Tobs, a.tau, tid);
                cta_sync<G>();
            }
            seq_window<N, G, PG>(&s_src[nw], a.orbit, a.tw, bufA1, bufE1, a.Tobs, a.tau, tid);
            if (tid == PG && nxt_ok) o1(theta_p + 8, s_src[nw ^ 1]);   // the next proposal's record, one ahead
            cp_async_wait<0>();
            cta_sync<G>();
            have = nxt_ok;
            if (cached) ns ^= 1;
            // ---- the five sums of Eq. 5 against the staged r' (buffers: 0 = old o, 1 = new a)
            const int64_t kmin_o = cached ? t.k_first + s_koff[k] : s_src[0].kmin;
            const int64_t j0o = kmin_o - t.k_first;   // staged bin of window bin 0, old and new
            const int64_t j0a = s_src[nw].kmin - t.k_first;
            const int64_t shift = s_src[nw].kmin - kmin_o;
            double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};   // aa, ra, ao, oo, ro
#pragma unroll
            for (int m = 0; m < S; m++) {
                const int j = tid + G * m;
                int64_t i = j0a + j;
                if (i >= 0 && i < t.n_stage) {
                    const cx ha = bufA1[pad_idx<N>(j)], he = bufE1[pad_idx<N>(j)];
                    const cx ra = sRA[i], re = sRE[i];
                    const double wa = sWA[i], we = sWE[i];
                    v[0] += wa * (ha.re * ha.re + ha.im * ha.im) + we * (he.re * he.re + he.im * he.im);
                    v[1] += wa * (ra.re * ha.re + ra.im * ha.im) + we * (re.re * he.re + re.im * he.im);
                    const int64_t jo = j + shift;
                    if (jo >= 0 && jo < N) {
                        const cx oa = bufA0[pad_idx<N>((int)jo)], oe = bufE0[pad_idx<N>((int)jo)];
                        v[2] += wa * (ha.re * oa.re + ha.im * oa.im) + we * (he.re * oe.re + he.im * oe.im);
                    }
                }
                i = j0o + j;
                if (i >= 0 && i < t.n_stage) {
                    const cx oa = bufA0[pad_idx<N>(j)], oe = bufE0[pad_idx<N>(j)];
                    const cx ra = sRA[i], re = sRE[i];
                    const double wa = sWA[i], we = sWE[i];
                    v[3] += wa * (oa.re * oa.re + oa.im * oa.im) + we * (oe.re * oe.re + oe.im * oe.im);
                    v[4] += wa * (ra.re * oa.re + ra.im * oa.im) + we * (re.re * oe.re + re.im * oe.im);
                }
            }
            group_reduce<G, 5>(v, s_red, tid);
            if (tid == 0) {
                const double norm = 4.0 / a.Tobs;
                const double dl = -0.5 * norm * (v[0] + v[3] - 2.0 * v[2] - 2.0 * v[1] + 2.0 * v[4]);
                const double lq = GEN ? s_glq[nw] : a.prop_logq[ip], lu = GEN ? s_glu[nw] : a.prop_logu[ip];
                const int acc = t.beta * dl + lq >= lu ? 1 : 0;
                a.dlnL_out[ip] = dl;
                a.accepted_out[ip] = (uint8_t)acc;
                s_acc = acc;
            }
            cta_sync<G>();
            if (s_acc) {
                // r' += h(theta_k), then r' -= h(theta'_k) (two passes: the windows overlap), and the same change
                // to the stored residual (only bins inside the stored band exist)
#pragma unroll
                for (int m = 0; m < S; m++) {
                    const int j = tid + G * m;
                    const int64_t i = j0o + j;
                    const int64_t e = i_first + i;
                    if (i >= 0 && i < t.n_stage && e >= 0 && e < a.n_f) {
                        const cx oa = bufA0[pad_idx<N>(j)], oe = bufE0[pad_idx<N>(j)];
                        sRA[i] = {sRA[i].re + oa.re, sRA[i].im + oa.im};
                        sRE[i] = {sRE[i].re + oe.re, sRE[i].im + oe.im};
                        if (wb) {
                            red_add_f64(wA + 2 * e, oa.re);
                            red_add_f64(wA + 2 * e + 1, oa.im);
                            red_add_f64(wE + 2 * e, oe.re);
                            red_add_f64(wE + 2 * e + 1, oe.im);
                        }
                    }
                }
                cta_sync<G>();
#pragma unroll
                for (int m = 0; m < S; m++) {
                    const int j = tid + G * m;
                    const int64_t i = j0a + j;
                    const int64_t e = i_first + i;
                    if (i >= 0 && i < t.n_stage && e >= 0 && e < a.n_f) {
                        const cx ha = bufA1[pad_idx<N>(j)], he = bufE1[pad_idx<N>(j)];
                        sRA[i] = {sRA[i].re - ha.re, sRA[i].im - ha.im};
                        sRE[i] = {sRE[i].re - he.re, sRE[i].im - he.im};
                        if (wb) {
                            red_add_f64(wA + 2 * e, -ha.re);
                            red_add_f64(wA + 2 * e + 1, -ha.im);
                            red_add_f64(wE + 2 * e, -he.re);
                            red_add_f64(wE + 2 * e + 1, -he.im);
                        }
                    }
                }
                if (tid < 8) {                              // theta_j[k] <- theta'_k
                    const double v = theta_p[tid];
                    theta_k[tid] = v;
                    if (gen_cached) s_theta[k][tid] = v;
                }
                if (gen_cached && tid == 0) s_redo = k;
                if (cached) {                               // and its window replaces the cached one
                    if (tid == 0) s_koff[k] = (int32_t)(s_src[nw].kmin - t.k_first);
#pragma unroll
                    for (int m = 0; m < S; m++) {
                        const int j = tid + G * m;
                        cache[((size_t)k * 2 + 0) * N + j] = bufA1[pad_idx<N>(j)];
                        cache[((size_t)k * 2 + 1) * N + j] = bufE1[pad_idx<N>(j)];
                    }
                }
            }
            cta_sync<G>();   // r', s_src, the waveform buffers and theta_j are reused by the next proposal
        }
    }
}
