// gb_temper.cuh -- Algorithm 2 of the paper as a kernel (Eq. D2).
// Included by gbfit.cu inside its anonymous namespace, after slow_part / fft_store / group_reduce.
//
// One CTA owns one sub-band's temperature ladder.  From the hottest pair down, chains i = t and j = t-1 propose to
// exchange the source sets they hold: the CTA builds delta = sum_{S_i} h - sum_{S_j} h on the staged bins in shared
// memory (one slow part + FFT per source, accumulated with its sign), reduces <delta|delta> and <r|delta> against
// both chains' residuals and PSD rows (read through L2), and thread 0 decides beta_i D_i + beta_j D_j >= logu
// with D_i = -1/2 <d|d>_i - <r_i|d>_i, D_j = -1/2 <d|d>_j + <r_j|d>_j.  An accepted exchange swaps the holders and
// (write_back) adds +-delta to the two stored residuals with FP64 atomics; the next pair then reads the updated
// residual of chain t-1 (the atomics resolve in L2, the reads are ld.global.cg after a fence and a barrier).
#pragma once

constexpr int kMaxLadder = 64;

struct TemperArgs {
    const gb_temper_task* tasks;
    int64_t n_tasks;
    const double* params;
    const int32_t* chain_walker;
    const double* chain_beta;
    const int32_t* chain_set_begin;
    const int32_t* chain_set_n;
    const double* chain_logu;
    int32_t* perm_out;
    uint8_t* accepted_out;
    double* dlnl_out;
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
    cx* cache;               // [gridDim.x][kTemperCacheChains][2][max_stage] summed windows of each chain's initial set
};

// Set-sum cache: a set takes part in up to two pairs (as S_j of pair (t+1, t), then as S_i of pair (t, t-1)) and only the
// SUM of its windows on the staged bins is ever needed.  Ladders of at most this many chains compute every chain's sum
// once into a per-CTA scratch area in global memory (L2 / HBM) and form delta = H_i - H_j from there: 95 instead of 171
// waveforms for a ladder of 10 chains with 9-10 sources each.
constexpr int kTemperCacheChains = 32;

template <int N>
constexpr size_t temper_smem_bytes(int max_stage) {
    return (size_t)padded_len<N>() * sizeof(cx) * 2 + (size_t)max_stage * 32;
}

// resident CTAs per SM the register allocation aims at: what shared memory allows at the usual stage of 3 N bins
template <int N>
constexpr int temper_min_blocks() { return N == 128 ? 6 : N == 256 ? 6 : N == 512 ? 3 : 1; }

template <int N, int GM>
__global__ void __launch_bounds__(Plan<N>::G * GM, temper_min_blocks<N>()) gb_temper_kernel(TemperArgs a) {
    constexpr int PG = Plan<N>::G;   // FFT group: the first PG threads
    constexpr int G = PG * GM;       // threads of the CTA
    constexpr int S = N / G;
    constexpr int PN = padded_len<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx* bufA = reinterpret_cast<cx*>(smem_raw);
    cx* bufE = bufA + PN;
    cx* dA = bufE + PN;                 // delta on the staged bins
    cx* dE = dA + a.max_stage;
    __shared__ __align__(16) SrcConst s_src[2];   // the source being generated and the next one (step O1 runs one source ahead)
    __shared__ double s_red[(G / 32) * 4 + 1];
    __shared__ int s_holder[kMaxLadder];
    __shared__ int s_acc;
    const int tid = threadIdx.x;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    const size_t nf = (size_t)a.n_f;

    for (int64_t it = blockIdx.x; it < a.n_tasks; it += gridDim.x) {
        const gb_temper_task t = a.tasks[it];
        // odd/even cold-chain buffers (Alg. 2 as printed): every chain's residual is its walker's row minus
        // the set it holds (formed below from the set sums); only an exchange with the cold chain is written, to write_walker
        const bool oddeven = (t.write_back & GB_TEMPER_ODD_EVEN) != 0;
        const bool wb = (t.write_back & GB_TEMPER_WRITE_BACK) != 0;
        bool ok = t.n_t >= 0 && t.n_t <= kMaxLadder && t.n_stage >= 0 && t.n_stage <= a.max_stage;
        if (oddeven) ok = ok && t.n_t <= kTemperCacheChains && a.cache != nullptr &&
                          (!wb || (t.write_walker >= 0 && t.write_walker < a.n_walkers));
        for (int q = 0; ok && q < t.n_t; q++) {
            const int w = a.chain_walker[t.chain_begin + q];
            ok = w >= 0 && w < a.n_walkers && a.chain_set_n[t.chain_begin + q] >= 0;
            if (ok) {
                const int row = a.walker_psd ? a.walker_psd[w] : (a.n_psd == 1 ? 0 : w);
                ok = row >= 0 && row < a.n_psd;
            }
        }
        for (int q = tid; q < t.n_t; q += G) {
            const int c = t.chain_begin + q;
            if (q < kMaxLadder) s_holder[q] = q;
            a.perm_out[c] = q;
            a.accepted_out[c] = 0;
            a.dlnl_out[2 * c] = a.dlnl_out[2 * c + 1] = (ok || q == 0) ? 0.0 : nan;
        }
        if (!ok) {
            if (tid == 0) atomicOr(a.errflag, 1);
            continue;
        }
        cta_sync<G>();
        const int64_t i_first = t.k_first - a.k_lo;
        // dA, dE += sign * (sum of the windows of the set held at chain entry `src`), on the staged bins.
        // Step O1 (one thread, ~1500 cycles) runs one source ahead: while the first PG threads transform source s, thread PG
        // -- idle otherwise -- works out the record of source s + 1 (the next source of the set, else `next_first`: the first
        // source of the set that the caller sums next) into the other half of s_src.
        constexpr bool kAhead = GM > 1;
        int slot = 0;
        bool have = false;   // s_src[slot] already holds the record of the next source (uniform over the CTA)
        auto o1 = [&](const double* theta, SrcConst& dst) { seq_o1<N>(theta, a.Tobs, a.tau, a.Rmax, a.kmax, a.errflag, &dst); };
        auto add_set = [&](int src, double sign, const double* next_first) {
            const int n_set = a.chain_set_n[src];
            const double* set = a.params + 8 * (size_t)a.chain_set_begin[src];
            for (int sidx = 0; sidx < n_set; sidx++) {
                if (!have) {
                    if (tid == 0) o1(set + 8 * sidx, s_src[slot]);
                    cta_sync<G>();
                }
                const SrcConst* cur = &s_src[slot];
                const double* nxt = !kAhead ? nullptr : sidx + 1 < n_set ? set + 8 * (sidx + 1) : next_first;
                seq_window<N, G, PG>(cur, a.orbit, a.tw, bufA, bufE, a.Tobs, a.tau, tid);
                if (tid == PG && nxt) o1(nxt, s_src[slot ^ 1]);
                cta_sync<G>();
                const int64_t j0 = cur->kmin - t.k_first;
#pragma unroll
                for (int m = 0; m < S; m++) {
                    const int j = tid + G * m;
                    const int64_t i = j0 + j;
                    if (i >= 0 && i < t.n_stage) {
                        const cx ha = bufA[pad_idx<N>(j)], he = bufE[pad_idx<N>(j)];
                        dA[i] = {dA[i].re + sign * ha.re, dA[i].im + sign * ha.im};
                        dE[i] = {dE[i].re + sign * he.re, dE[i].im + sign * he.im};
                    }
                }
                cta_sync<G>();
                have = nxt != nullptr;
                slot ^= 1;
            }
        };
        // first source of the first non-empty set among chain entries [c, c_end), or NULL
        auto first_source = [&](int c, int c_end) -> const double* {
            for (; c < c_end; c++)
                if (a.chain_set_n[c] > 0) return a.params + 8 * (size_t)a.chain_set_begin[c];
            return nullptr;
        };
        auto zero_delta = [&]() {
            for (int i = tid; i < t.n_stage; i += G) {
                dA[i] = {0.0, 0.0};
                dE[i] = {0.0, 0.0};
            }
            cta_sync<G>();
        };
        cx* cache = a.cache ? a.cache + (size_t)blockIdx.x * kTemperCacheChains * 2 * a.max_stage : nullptr;
        const bool cached = cache != nullptr && t.n_t <= kTemperCacheChains && (t.n_t > 2 || oddeven);
        if (cached) {   // H_c = sum of the windows of chain c's initial set
            for (int c = 0; c < t.n_t; c++) {
                zero_delta();
                add_set(t.chain_begin + c, 1.0, first_source(t.chain_begin + c + 1, t.chain_begin + t.n_t));
                for (int i = tid; i < t.n_stage; i += G) {
                    cache[((size_t)c * 2 + 0) * a.max_stage + i] = dA[i];
                    cache[((size_t)c * 2 + 1) * a.max_stage + i] = dE[i];
                }
                cta_sync<G>();
            }
        }
        for (int q = t.n_t - 1; q >= 1; q--) {
            const int ci = t.chain_begin + q, cj = ci - 1;
            // ---- delta = sum over the set chain i holds - sum over the set chain j holds
            if (cached) {
                const cx* Hi = cache + (size_t)s_holder[q] * 2 * a.max_stage;
                const cx* Hj = cache + (size_t)s_holder[q - 1] * 2 * a.max_stage;
                // (four bins per thread in flight: the set sums come from L2 / HBM and a round trip per bin is the whole loop)
                for (int i0 = tid; i0 < t.n_stage; i0 += 4 * G) {
                    cx ai[4], ei[4], aj[4], ej[4];
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const int i = min(i0 + u * G, t.n_stage - 1);
                        ai[u] = Hi[i];
                        ei[u] = Hi[a.max_stage + i];
                        aj[u] = Hj[i];
                        ej[u] = Hj[a.max_stage + i];
                    }
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const int i = i0 + u * G;
                        if (i < t.n_stage) {
                            dA[i] = {ai[u].re - aj[u].re, ai[u].im - aj[u].im};
                            dE[i] = {ei[u].re - ej[u].re, ei[u].im - ej[u].im};
                        }
                    }
                }
                cta_sync<G>();
            } else {
                zero_delta();
                add_set(t.chain_begin + s_holder[q], 1.0, first_source(t.chain_begin + s_holder[q - 1], t.chain_begin + s_holder[q - 1] + 1));
                add_set(t.chain_begin + s_holder[q - 1], -1.0, nullptr);
            }
            // ---- <delta|delta> and <r|delta> for both chains, stored bins only
            const int wi = a.chain_walker[ci], wj = a.chain_walker[cj];
            const int rowi = a.walker_psd ? a.walker_psd[wi] : (a.n_psd == 1 ? 0 : wi);
            const int rowj = a.walker_psd ? a.walker_psd[wj] : (a.n_psd == 1 ? 0 : wj);
            double* rAi = a.resid + ((size_t)wi * 2 + 0) * nf * 2;
            double* rEi = a.resid + ((size_t)wi * 2 + 1) * nf * 2;
            double* rAj = a.resid + ((size_t)wj * 2 + 0) * nf * 2;
            double* rEj = a.resid + ((size_t)wj * 2 + 1) * nf * 2;
            const double* SAi = a.psd + ((size_t)rowi * 2 + 0) * nf;
            const double* SEi = a.psd + ((size_t)rowi * 2 + 1) * nf;
            const double* SAj = a.psd + ((size_t)rowj * 2 + 0) * nf;
            const double* SEj = a.psd + ((size_t)rowj * 2 + 1) * nf;
            const bool inv = a.psd_is_inverse != 0;
            double v[4] = {0.0, 0.0, 0.0, 0.0};   // dd_i, rd_i, dd_j, rd_j
            const cx* Hi = cached ? cache + (size_t)s_holder[q] * 2 * a.max_stage : nullptr;       // the set sums the two
            const cx* Hj = cached ? cache + (size_t)s_holder[q - 1] * 2 * a.max_stage : nullptr;   // chains hold
            // two bins per thread in flight (residual rows, weights and -- odd/even -- the set sums come from L2 / HBM)
            for (int i0 = tid; i0 < t.n_stage; i0 += 2 * G) {
                double2 rai[2], rei[2], raj[2], rej[2];
                double wai[2], wei[2], waj[2], wej[2];
                bool okb[2];
#pragma unroll
                for (int u = 0; u < 2; u++) {
                    const int i = i0 + u * G;
                    const int64_t e = i_first + i;
                    okb[u] = i < t.n_stage && e >= 0 && e < a.n_f;
                    const int64_t ec = okb[u] ? e : (i_first < 0 ? 0 : i_first >= a.n_f ? a.n_f - 1 : i_first);
                    rai[u] = __ldcg(reinterpret_cast<const double2*>(rAi + 2 * ec));
                    rei[u] = __ldcg(reinterpret_cast<const double2*>(rEi + 2 * ec));
                    raj[u] = __ldcg(reinterpret_cast<const double2*>(rAj + 2 * ec));
                    rej[u] = __ldcg(reinterpret_cast<const double2*>(rEj + 2 * ec));
                    wai[u] = SAi[ec];
                    wei[u] = SEi[ec];
                    waj[u] = SAj[ec];
                    wej[u] = SEj[ec];
                }
#pragma unroll
                for (int u = 0; u < 2; u++) {
                    if (!okb[u]) continue;
                    const int i = i0 + u * G;
                    const cx da = dA[i], de = dE[i];
                    const double na = da.re * da.re + da.im * da.im, ne = de.re * de.re + de.im * de.im;
                    {
                        double2 ra = rai[u], re = rei[u];
                        if (oddeven) {   // r_i = row - sum_{S_i} h
                            const cx ha = Hi[i], he = Hi[a.max_stage + i];
                            ra.x -= ha.re;  ra.y -= ha.im;  re.x -= he.re;  re.y -= he.im;
                        }
                        const double wa = inv ? wai[u] : 1.0 / wai[u], we = inv ? wei[u] : 1.0 / wei[u];
                        v[0] += wa * na + we * ne;
                        v[1] += wa * (ra.x * da.re + ra.y * da.im) + we * (re.x * de.re + re.y * de.im);
                    }
                    {
                        double2 ra = raj[u], re = rej[u];
                        if (oddeven) {
                            const cx ha = Hj[i], he = Hj[a.max_stage + i];
                            ra.x -= ha.re;  ra.y -= ha.im;  re.x -= he.re;  re.y -= he.im;
                        }
                        const double wa = inv ? waj[u] : 1.0 / waj[u], we = inv ? wej[u] : 1.0 / wej[u];
                        v[2] += wa * na + we * ne;
                        v[3] += wa * (ra.x * da.re + ra.y * da.im) + we * (re.x * de.re + re.y * de.im);
                    }
                }
            }
            group_reduce<G, 4>(v, s_red, tid);
            if (tid == 0) {
                const double norm = 4.0 / a.Tobs;
                const double Di = -0.5 * norm * v[0] - norm * v[1];
                const double Dj = -0.5 * norm * v[2] + norm * v[3];
                const int acc = a.chain_beta[ci] * Di + a.chain_beta[cj] * Dj >= a.chain_logu[ci] ? 1 : 0;
                a.accepted_out[ci] = (uint8_t)acc;
                a.dlnl_out[2 * ci] = Di;
                a.dlnl_out[2 * ci + 1] = Dj;
                s_acc = acc;
                if (acc) {
                    const int h = s_holder[q];
                    s_holder[q] = s_holder[q - 1];
                    s_holder[q - 1] = h;
                }
            }
            cta_sync<G>();
            if (s_acc && oddeven) {
                if (wb && q == 1) {   // the cold chain now holds S_i: its buffer of the band's own parity -= delta (:652-658)
                    double* wA = a.resid + ((size_t)t.write_walker * 2 + 0) * nf * 2;
                    double* wE = a.resid + ((size_t)t.write_walker * 2 + 1) * nf * 2;
                    for (int i = tid; i < t.n_stage; i += G) {
                        const int64_t e = i_first + i;
                        if (e < 0 || e >= a.n_f) continue;
                        const cx da = dA[i], de = dE[i];
                        red_add_f64(wA + 2 * e, -da.re);
                        red_add_f64(wA + 2 * e + 1, -da.im);
                        red_add_f64(wE + 2 * e, -de.re);
                        red_add_f64(wE + 2 * e + 1, -de.im);
                    }
                }
            } else if (s_acc && wb) {   // r_i += delta, r_j -= delta
                for (int i = tid; i < t.n_stage; i += G) {
                    const int64_t e = i_first + i;
                    if (e < 0 || e >= a.n_f) continue;
                    const cx da = dA[i], de = dE[i];
                    red_add_f64(rAi + 2 * e, da.re);
                    red_add_f64(rAi + 2 * e + 1, da.im);
                    red_add_f64(rEi + 2 * e, de.re);
                    red_add_f64(rEi + 2 * e + 1, de.im);
                    red_add_f64(rAj + 2 * e, -da.re);
                    red_add_f64(rAj + 2 * e + 1, -da.im);
                    red_add_f64(rEj + 2 * e, -de.re);
                    red_add_f64(rEj + 2 * e + 1, -de.im);
                }
                __threadfence();
            }
            cta_sync<G>();
        }
        for (int q = tid; q < t.n_t; q += G) a.perm_out[t.chain_begin + q] = s_holder[q];
        cta_sync<G>();
    }
}
