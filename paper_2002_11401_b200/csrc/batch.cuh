// batch.cuh -- exact batched flips for the relax loop.  Included by flatspin.cu only.
//
// The relaxation of PAPER.md:122-124 is sequential by definition: "flip the spin where ... Eq. (5) is
// greatest", repeat ("switching is sequential", "the magnet experiencing the highest
// effective field ... is the first to switch").  k_relax does exactly that, one dependent chain per flip on
// one SM.  This kernel produces the IDENTICAL flip sequence many flips at a time on all SMs:
//
//  * A flip of spin k reads and writes only the closed neighbourhood N[k] = nbr(k) U {k} (Eq. 3 is a sum
//    over the neighbourhood).  Flips whose closed neighbourhoods are disjoint commute in
//    state; only their ORDER in the log is global.
//  * Per round: the candidates with margin above a threshold theta ("seeds", at most P of them) are taken.
//    Seeds whose closed neighbourhoods overlap are joined into components (label propagation over the
//    claim table `owner`).  One warp per component runs the sequential rule LOCALLY: repeatedly flip the
//    local arg-max among the component's seeds and the spins its own flips have made switchable, while
//    that arg-max is above theta, claiming the closed neighbourhood of every spin it flips.  Inside a
//    region nobody else touches, the local order IS the global order restricted to that region.
//  * The global order of independent local sequences is the greedy merge "always take the largest head".
//    That equals a sort by the EFFECTIVE key = running minimum of the actual keys along the local
//    sequence (an element cannot come before its predecessors; once a low head is taken, its higher
//    successors follow at once), ties by the index of the minimum's spin, then by position.
//  * Everything not simulated this round has key <= theta.  A component that cannot continue (it would
//    touch a spin another component owns, or ran out of room) posts a "blocker" at the effective key of
//    the element it could not do.  The CUT is the earliest blocker (or theta): elements before the cut
//    are exactly the next flips of the sequential process and are committed, in merged order, to the flip
//    log; elements after it are undone from their undo records (old h_dip, margin, spin restored bit
//    for bit) and simply happen again in a later round.
//
// Exactness does not depend on how races for claims resolve: any committed set is a prefix of the true
// sequence.  When few candidates remain the kernel rebuilds the leaf maxima and k_relax finishes the tail.
// A CPU prototype of this rule reproduced the sequential log on configs 3 and 4 (full size: 2,002,000 flips
// in 1,993 rounds); on the GPU the parity suite compares the logs with the oracle's, as before.
#pragma once

constexpr int BT_THREADS = 1024;
constexpr int BT_NB = 2048;            // histogram bins
constexpr int BT_PMAX = 4096;          // seeds per round: a seed slot fits 12 bits of the claim word
constexpr int BT_LMAX = 16;            // flips per component per round
constexpr int BT_EMAX = 8;             // distinct conflicting owners recorded per seed

struct BatchSeed { mkey_t key; int idx; int pad; };
struct BatchElem { mkey_t ev; int ei; int k; };                    // effective key (ev, ei); position = array index
struct BatchUndo { double2 hd; double M; int idx; int pad; };
struct BatchCommit { mkey_t nev; unsigned long long lo; int k; int pad; };   // sort key (~ev, ei << 32 | pos), ascending
struct BatchBlock { mkey_t ev; int ei; int pos; };

struct BatchCtl {                      // zeroed once at creation; every launch leaves it clean for the next one
    unsigned bar[2];                   // grid barrier counters (monotone within a launch), alternating between launches
    unsigned bail;                     // 1 = exact ties defeated the threshold search in the last launch
    unsigned round_base;               // rounds of all launches so far: the claim tag of a round is unique across launches
    unsigned launch;                   // launches that used the barrier so far (their parity picks the counter)
    unsigned n_list;                   // entries of the candidate list (this launch)
    unsigned n_seeds[4], n_commit[4], n_block[4];      // rotating per-round counters
    unsigned long long n_cand[3];
    unsigned hist[3][BT_NB];           // rotating histograms (one per pass)
    long long flips, rounds, undone, blockers;         // results / statistics of this launch
    long long prof[12];                // FS_BATCH_PROFILE: nanoseconds per phase (CTA 0), accumulated
};

struct BatchArgs {
    int64_t N; int Kp, LBshift, nblk; Astroid ast; long long log_cap;
    const int* nbr; const double2* wT; const double* ihc; int8_t* s; double2* hdip; const double2* hfix; double* M;
    double* bval; int* bidx; int* flog; Counters* ctr;
    const int* cellidx; sgcell_t* sgrid;
    // scratch
    BatchCtl* ctl; unsigned* owner; BatchSeed* seeds; unsigned short* edges; unsigned char* ecount;
    int* npos; BatchElem* elems; BatchUndo* undo; BatchBlock* blocks; BatchCommit* clist;
    int* cand; unsigned* cbits;        // candidate list: every spin with margin > 1 is in it (dead entries stay), bit = listed
    int P, seq_threshold, min_commit, max_chain;
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// all CTAs are co-resident (cooperative launch): counter barrier, one atomic per CTA
__device__ __forceinline__ void grid_bar(unsigned* bar, unsigned& epoch) {
    __syncthreads();
    epoch += gridDim.x;
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        while (ld_acquire_u32(bar) < epoch) {}
        __threadfence();
    }
    __syncthreads();
}

// monotone map of d = key - KEY_ONE - 1 >= 0 to a bin: position of the top bit and the 5 bits below it
__device__ __forceinline__ int log_bin(unsigned long long d) {
    if (d < 64) return (int)d;                                    // bins 0..63: exact
    int e = 63 - __clzll((long long)d);                           // >= 6
    return (e - 4) * 32 + (int)((d >> (e - 5)) & 31);             // e = 6 -> 64..95; e = 63 -> 1888..1919
}
__device__ __forceinline__ unsigned long long log_bin_lo(int b) { // smallest d of bin b
    if (b < 64) return (unsigned long long)b;
    int e = (b >> 5) + 4, m = b & 31;
    return (unsigned long long)(32 + m) << (e - 5);
}

// is element (ev, ei, pos) before (bv, bi, bp) in the merged order?  key descending, index ascending, position ascending
__device__ __forceinline__ bool bt_before(mkey_t ev, int ei, int pos, mkey_t bv, int bi, int bp) {
    return ev > bv || (ev == bv && (ei < bi || (ei == bi && pos < bp)));
}

#ifdef FS_BATCH_PROFILE
__device__ __forceinline__ long long bt_now() { long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#define BT_PROF(slot) do { if (gtid == 0) { const long long t_ = bt_now(); g->prof[slot] += t_ - tprof; tprof = t_; } } while (0)
#else
#define BT_PROF(slot)
#endif

__global__ void __launch_bounds__(BT_THREADS, 1) k_relax_batch(BatchArgs a) {
    __shared__ unsigned sh_hist[BT_NB];
    __shared__ int sh_label[BT_PMAX];
    __shared__ unsigned sh_cnt[BT_PMAX];
    __shared__ unsigned sh_scan[BT_THREADS / 32];
    __shared__ int sh_bstar;
    __shared__ unsigned sh_sel, sh_below;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthreads = gridDim.x * BT_THREADS;
    const int gtid = blockIdx.x * BT_THREADS + tid;
    const int gwarp = gtid >> 5, nwarps = nthreads >> 5;
    const int64_t N = a.N;
    const int Kp = a.Kp;
    BatchCtl* g = a.ctl;
    // k_scan (finalize) left the number of switchable spins: with only a few, k_relax does it alone (uniform exit,
    // nothing touched)
    if (__ldcg(&a.ctr[0].n_switchable) <= (long long)a.seq_threshold) {
        if (blockIdx.x == 0 && threadIdx.x == 0) a.ctr[0].batch_flips = 0;
        return;
    }
    const unsigned parity = __ldcg(&g->launch) & 1u;
    unsigned* const bar = &g->bar[parity];
    unsigned epoch = 0;
    unsigned round_base = __ldcg(&g->round_base);
    if (round_base > 0xF0000u) {                        // claim tags nearly used up: wipe the claim table
        for (int64_t i = blockIdx.x * (int64_t)BT_THREADS + threadIdx.x; i < a.N; i += (int64_t)gridDim.x * BT_THREADS) a.owner[i] = 0xFFFFFFFFu;
        grid_bar(bar, epoch);
        round_base = 0;
    }
    long long nflips = 0, rounds = 0, undone = 0, nblockers = 0;
    int rot = 0;                                        // rotating counter slot of this round
    unsigned npass = 0;                                 // histogram passes so far (buffer = npass % 3)
    bool any_flip = false;
    int lean = 0;                                       // consecutive rounds that committed fewer than min_commit flips

    // ---- candidate list: every spin with margin > 1 (one pass over M per launch; the rounds then touch only the list).
    // Invariant at the start of every round: {i : M_i > 1} is a subset of the list.  Spins whose margin falls to <= 1
    // stay as dead entries (skipped by their margin); spins that become switchable are appended when a round
    // commits the flip that touched them.
    for (int64_t wd = gtid; wd < (N + 31) / 32; wd += nthreads) a.cbits[wd] = 0u;
    if (gtid == 0) g->n_list = 0u;
    grid_bar(bar, epoch);
    for (int64_t i0 = (int64_t)gwarp * 32; i0 < N; i0 += (int64_t)nwarps * 32) {
        const int64_t i = i0 + lane;
        const bool c = i < N && __ldcg(a.M + i) > 1.0;
        const unsigned m = __ballot_sync(0xffffffffu, c);
        if (m) {
            unsigned base = 0;
            if (lane == 0) { base = atomicAdd(&g->n_list, (unsigned)__popc(m)); a.cbits[i0 >> 5] = m; }   // word i0/32 is this warp's
            base = __shfl_sync(0xffffffffu, base, 0);
            if (c) a.cand[base + __popc(m & ((1u << lane) - 1u))] = (int)i;
        }
    }
    grid_bar(bar, epoch);
#ifdef FS_BATCH_PROFILE
    long long tprof = bt_now();
#endif
    for (;; ++rounds) {
        // newer rounds win an atomicMin on the claim word.  Tag 0xFFFFF is never issued: it is the tag field of 0xFFFFFFFF,
        // the "unowned" word the claim table is filled with (round_base + rounds <= 0xF0000 + 0xFFF0, so tag >= 0xE)
        const unsigned tag = 0xFFFFEu - (round_base + (unsigned)rounds);
        if (rounds >= 0xFFF0) break;
        // ================= phase 1: threshold theta such that <= P candidates have key > theta ==============
        // One pass over all margins builds a histogram of log-spaced bins of (key - 1); theta is the lower edge
        // of the lowest bin b* whose suffix count still fits P.  If that takes fewer than P/4 seeds although the
        // next bin is populated (one bin holds more than P candidates), that bin is split linearly by a further
        // pass.  Every CTA derives the same theta from the same global histogram.
        unsigned long long lo = 0, hi = 0; int shift = -1;           // shift < 0: log bins; else linear bins over (lo, hi]
        unsigned long long theta = KEY_ONE; unsigned above = 0;      // `above` = candidates with key > hi (already selected)
        unsigned long long ncand_total = 0;
        bool have_theta = false, quit = false;
        const unsigned P = (unsigned)a.P;
        const int nl = (int)__ldcg(&g->n_list);
        for (int refine = 0; refine < 8 && !have_theta; ++refine, ++npass) {
            const int hb = (int)(npass % 3);
            for (int b = tid; b < BT_NB; b += BT_THREADS) sh_hist[b] = 0;
            __syncthreads();
            unsigned my_cand = 0;
            for (int j = gtid; j < nl; j += nthreads) {
                const mkey_t key = margin_key(__ldcg(a.M + a.cand[j]));
                if (key > KEY_ONE) {
                    ++my_cand;
                    if (shift < 0) atomicAdd(&sh_hist[log_bin(key - KEY_ONE - 1)], 1u);
                    else if (key > lo && key <= hi)
                        atomicAdd(&sh_hist[(int)min((unsigned long long)(BT_NB - 1), (key - lo - 1) >> shift)], 1u);
                }
            }
            __syncthreads();
            for (int b = tid; b < BT_NB; b += BT_THREADS) if (sh_hist[b]) atomicAdd(&g->hist[hb][b], sh_hist[b]);
            if (shift < 0) {
                my_cand = __reduce_add_sync(0xffffffffu, my_cand);
                if (lane == 0 && my_cand) atomicAdd(&g->n_cand[hb], (unsigned long long)my_cand);
            }
            grid_bar(bar, epoch);
            if (blockIdx.x == 0) {                                   // the buffer of the previous pass: everyone has read it
                const int zb = (hb + 2) % 3;
                for (int b = tid; b < BT_NB; b += BT_THREADS) g->hist[zb][b] = 0;
                if (tid == 0) g->n_cand[zb] = 0;
            }
            if (shift < 0) {
                ncand_total = __ldcg(&g->n_cand[hb]);
                if (ncand_total <= (unsigned long long)a.seq_threshold) { quit = true; ++npass; break; }   // the tail belongs to k_relax
            }
            // suffix counts S(b) = above + sum_{b' >= b} hist[b']; thread t owns bins 2t and 2t+1
            const unsigned h0 = __ldcg(&g->hist[hb][2 * tid]), h1 = __ldcg(&g->hist[hb][2 * tid + 1]);
            const unsigned mine = h0 + h1;
            unsigned incl = mine;                                    // inclusive suffix sum over the threads >= tid
            for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_down_sync(0xffffffffu, incl, o); if (lane + o < 32) incl += t; }
            if (lane == 0) sh_scan[warp] = incl;
            if (tid == 0) { sh_bstar = -1; }
            __syncthreads();
            if (warp == 0) {
                const unsigned v = sh_scan[lane]; unsigned inc2 = v;
                for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_down_sync(0xffffffffu, inc2, o); if (lane + o < 32) inc2 += t; }
                sh_scan[lane] = inc2 - v;                           // total of the warps above this one
            }
            __syncthreads();
            const unsigned S1 = above + sh_scan[warp] + (incl - mine) + h1;      // S(2t+1)
            const unsigned S0 = S1 + h0;                                          // S(2t)
            const unsigned hm1 = tid > 0 ? __ldcg(&g->hist[hb][2 * tid - 1]) : 0u;
            // b* = smallest bin with S(b*) <= P (S is non-increasing); b* = NB if even the top bin is too full
            if (S1 <= P && S0 > P) { sh_bstar = 2 * tid + 1; sh_sel = S1; sh_below = h0; }
            else if (S0 <= P && (tid == 0 || S0 + hm1 > P)) { sh_bstar = 2 * tid; sh_sel = S0; sh_below = hm1; }
            if (tid == BT_THREADS - 1 && S1 > P) { sh_bstar = BT_NB; sh_sel = above; sh_below = h1; }
            __syncthreads();
            const int bstar = sh_bstar; const unsigned sel = sh_sel, below = sh_below;
            auto edge = [&](int b) -> unsigned long long {           // keys of bin b are > edge(b) (and <= edge(b + 1))
                if (shift < 0) return b >= 1920 ? ~0ull : KEY_ONE + log_bin_lo(b);
                return b >= BT_NB ? hi : lo + ((unsigned long long)b << shift);
            };
            theta = edge(bstar);
            if (bstar == 0 || sel >= P / 4 || below == 0 || refine == 7) {
                have_theta = sel > 0 || bstar == 0; if (!have_theta) quit = true;
                ++npass; break;
            }
            // split bin b* - 1
            const unsigned long long nlo = edge(bstar - 1), nhi = theta;
            if (nhi - nlo <= 1) { have_theta = sel > 0; if (!have_theta) quit = true; ++npass; break; }   // one key value: exact ties
            lo = nlo; hi = nhi; above = sel;
            const unsigned long long range = hi - lo - 1;            // bins index (key - lo - 1) in [0, range]
            shift = max(0, 64 - __clzll((long long)range) - 11);
        }
        if (quit || !have_theta) {
            if (ncand_total > (unsigned long long)a.seq_threshold && gtid == 0) g->bail = 1;       // exact ties defeat the search
            break;
        }
        BT_PROF(0);
        // ================= phase 2: seeds = candidates with key > theta ====================================
        BatchSeed* seeds = a.seeds;
        for (int j0 = gwarp * 32; j0 < nl; j0 += nwarps * 32) {
            const int j = j0 + lane;
            const int i = j < nl ? a.cand[j] : -1;
            const mkey_t key = i >= 0 ? margin_key(__ldcg(a.M + i)) : 0ull;
            const bool sel = key > theta;
            const unsigned m = __ballot_sync(0xffffffffu, sel);
            if (m) {
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(&g->n_seeds[rot], (unsigned)__popc(m));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (sel) {
                    const unsigned slot = base + __popc(m & ((1u << lane) - 1u));
                    if (slot < BT_PMAX) seeds[slot] = BatchSeed{key, i, 0};
                }
            }
        }
        grid_bar(bar, epoch);
        const int n_seeds = (int)min(__ldcg(&g->n_seeds[rot]), (unsigned)BT_PMAX);
        if (blockIdx.x == 0 && tid == 0) {                                       // counters two rounds ahead
            const int z = (rot + 2) & 3;
            g->n_seeds[z] = 0; g->n_commit[z] = 0; g->n_block[z] = 0;
        }
        BT_PROF(1);
        // ================= phase 3: claims.  owner[t] = min over seeds claiming t of (tag, slot) ============
        for (int r = gwarp; r < n_seeds; r += nwarps) {
            const int k = seeds[r].idx;
            const int* rowk = a.nbr + (int64_t)k * Kp;
            const unsigned word = (tag << 12) | (unsigned)r;
            for (int t = lane; t <= Kp; t += 32) {
                const int i = (t == Kp) ? k : rowk[t];
                if (i >= 0) atomicMin(a.owner + i, word);
            }
        }
        grid_bar(bar, epoch);
        BT_PROF(2);
        // ================= phase 4: conflict edges (seed r shares a spin with the seed that owns it) ========
        for (int r = gwarp; r < n_seeds; r += nwarps) {
            const int k = seeds[r].idx;
            const int* rowk = a.nbr + (int64_t)k * Kp;
            int ne = 0;
            for (int t0 = 0; t0 <= Kp; t0 += 32) {
                const int t = t0 + lane;
                const int i = (t > Kp) ? -1 : ((t == Kp) ? k : rowk[t]);
                int o = -1;
                if (i >= 0) o = (int)(__ldcg(a.owner + i) & 0xFFFu);
                unsigned m = __ballot_sync(0xffffffffu, o >= 0 && o != r);
                while (m) {
                    const int src = __ffs(m) - 1;
                    const int oo = __shfl_sync(0xffffffffu, o, src);
                    m &= ~__ballot_sync(0xffffffffu, o == oo);                   // all lanes that saw the same owner
                    if (ne < BT_EMAX) { if (lane == 0) a.edges[r * BT_EMAX + ne] = (unsigned short)oo; }
                    ++ne;
                }
            }
            if (lane == 0) a.ecount[r] = (unsigned char)(ne > BT_EMAX ? 0xFF : ne);
        }
        grid_bar(bar, epoch);
        BT_PROF(3);
        // ================= phase 5: components (every CTA computes the same labels in shared memory) ========
        for (int r = tid; r < n_seeds; r += BT_THREADS) { sh_label[r] = r; sh_cnt[r] = __ldcg(a.ecount + r); }   // edge counts cached
        __syncthreads();
        for (;;) {
            int changed = 0;
            for (int r = tid; r < n_seeds; r += BT_THREADS) {
                const unsigned ec = sh_cnt[r];
                if (!ec) continue;                                               // most seeds conflict with nobody
                const int n = ec == 0xFF ? BT_EMAX : (int)ec;
                for (int e = 0; e < n; ++e) {
                    const int o = __ldcg(a.edges + r * BT_EMAX + e);
                    const int lr = sh_label[r], lo_ = sh_label[o], m = min(lr, lo_);
                    if (lr != m) { atomicMin(&sh_label[r], m); changed = 1; }
                    if (lo_ != m) { atomicMin(&sh_label[o], m); changed = 1; }
                }
            }
            __syncthreads();
            for (int r = tid; r < n_seeds; r += BT_THREADS) {
                const int l = sh_label[r], ll = sh_label[l];
                if (ll < l) { atomicMin(&sh_label[r], ll); changed = 1; }
            }
            if (!__syncthreads_or(changed)) break;
        }
        for (int r = tid; r < n_seeds; r += BT_THREADS) sh_cnt[r] = 0;
        __syncthreads();
        for (int r = tid; r < n_seeds; r += BT_THREADS) atomicAdd(&sh_cnt[sh_label[r]], 1u);     // members per component
        __syncthreads();
        BT_PROF(4);
        // ================= phase 6: one warp per component runs the sequential rule locally ==================
        for (int r = gwarp; r < n_seeds; r += nwarps) {
            if (sh_label[r] != r) continue;                                      // not a leader
            const int leader = r;
            int a_idx = -1; mkey_t a_key = 0ull;                                 // active set: one entry per lane
            int na = 0; bool blocked = false;
            mkey_t topk = 0ull; int topi = 0x7fffffff;
            if (sh_cnt[r] == 1) {
                const BatchSeed sd = seeds[r];
                if (lane == 0) { a_idx = sd.idx; a_key = sd.key; }
                na = 1; blocked = __ldcg(a.ecount + r) == 0xFF;
                topk = sd.key; topi = sd.idx;
            } else {
                for (int base = 0; base < n_seeds; base += 32) {
                    const int q = base + lane;
                    const bool mem = q < n_seeds && sh_label[q] == leader;
                    unsigned m = __ballot_sync(0xffffffffu, mem);
                    while (m) {
                        const int q2 = base + __ffs(m) - 1; m &= m - 1;
                        const BatchSeed sd = seeds[q2];
                        if (__ldcg(a.ecount + q2) == 0xFF) blocked = true;
                        if (na < 32) { if (lane == na) { a_idx = sd.idx; a_key = sd.key; } }
                        else blocked = true;
                        ++na;
                        if (sd.key > topk || (sd.key == topk && sd.idx < topi)) { topk = sd.key; topi = sd.idx; }
                    }
                }
            }
            int pos = 0;
            mkey_t ev = ~0ull; int ei = -1;
            bool post = false; mkey_t pv = 0; int pi = 0, pp = 0;               // blocker to post
            if (blocked) { post = true; pv = topk; pi = topi; pp = 0; }
            while (!blocked) {
                mkey_t bk = a_idx >= 0 ? a_key : 0ull; int k = a_idx >= 0 ? a_idx : 0x7fffffff;
                warp_argmax_key(bk, k);
                if (!(bk > theta)) break;                                        // what is left is <= theta
                if (bk < ev || (bk == ev && k > ei)) { ev = bk; ei = k; }       // running minimum in flip order
                if (pos >= a.max_chain) { post = true; pv = ev; pi = ei; pp = pos; break; }
                const int* rowk = a.nbr + (int64_t)k * Kp;
                // claim the closed neighbourhood
                bool ok = true;
                for (int t = lane; t <= Kp; t += 32) {
                    const int i = (t == Kp) ? k : rowk[t];
                    if (i < 0) continue;
                    unsigned o = __ldcg(a.owner + i);
                    for (;;) {
                        if (o != 0xFFFFFFFFu && (o >> 12) == tag) { ok &= sh_label[o & 0xFFFu] == leader; break; }   // an unowned word always takes the CAS
                        const unsigned prev = atomicCAS(a.owner + i, o, (tag << 12) | (unsigned)leader);
                        if (prev == o) break;
                        o = prev;
                    }
                }
                if (!__all_sync(0xffffffffu, ok)) { post = true; pv = ev; pi = ei; pp = pos; break; }
                // flip k: h_i -= 2 s_k,old alpha g_ik over nbr(k) (Eq. 3 linear in s_k), new margins, undo records
                const double2* wTk = a.wT + (int64_t)k * Kp;
                const int s_old = __ldcg(a.s + k);
                const double two_s = 2.0 * (double)s_old;
                BatchUndo* und = a.undo + ((int64_t)leader * BT_LMAX + pos) * (Kp + 1);
                bool overflow = false;
                for (int t0 = 0; t0 <= Kp; t0 += 32) {
                    const int t = t0 + lane;
                    const int i = (t > Kp) ? -1 : ((t == Kp) ? k : rowk[t]);
                    mkey_t nk = 0ull; bool was = false;
                    if (i >= 0) {
                        double2 hd = __ldcg(a.hdip + i); const double2 hf = a.hfix[i];
                        const double mo = __ldcg(a.M + i);
                        double si = (double)__ldcg(a.s + i); const double ih = a.ihc[i];
                        und[t] = BatchUndo{hd, mo, i, 0};
                        if (t == Kp) si = -(double)s_old;
                        else {
                            const double2 wt = wTk[t];
                            hd.x -= two_s * wt.x;
                            hd.y -= two_s * wt.y;
                            a.hdip[i] = hd;
                        }
                        const double m = margin(hd.x + hf.x, hd.y + hf.y, si, ih, a.ast);
                        a.M[i] = m;
                        nk = margin_key(m); was = mo > 1.0;
                    } else if (t <= Kp) und[t] = BatchUndo{make_double2(0.0, 0.0), 0.0, -1, 0};
                    // active set: refresh the entries of touched spins, insert new candidates
                    unsigned need = __ballot_sync(0xffffffffu, i >= 0 && (nk > KEY_ONE || was));
                    while (need) {
                        const int src = __ffs(need) - 1; need &= need - 1;
                        const int bi = __shfl_sync(0xffffffffu, i, src);
                        const mkey_t bkey = __shfl_sync(0xffffffffu, nk, src);
                        const unsigned found = __ballot_sync(0xffffffffu, a_idx == bi);
                        if (found) {
                            if (lane == __ffs(found) - 1) { if (bkey > KEY_ONE) a_key = bkey; else a_idx = -1; }
                        } else if (bkey > KEY_ONE) {
                            const unsigned fr = __ballot_sync(0xffffffffu, a_idx < 0);
                            if (!fr) overflow = true;
                            else if (lane == __ffs(fr) - 1) { a_idx = bi; a_key = bkey; }
                        }
                    }
                }
                if (lane == 0) {
                    a.s[k] = (int8_t)(-s_old);
                    a.elems[(int64_t)leader * BT_LMAX + pos] = BatchElem{ev, ei, k};
                }
                ++pos;
                __syncwarp();
                if (overflow) { post = true; pv = ev; pi = ei; pp = pos; break; }
            }
            if (lane == 0) {
                a.npos[leader] = pos;
                if (post) {
                    const unsigned slot = atomicAdd(&g->n_block[rot], 1u);
                    if (slot < BT_PMAX) a.blocks[slot] = BatchBlock{pv, pi, pp};
                }
            }
        }
        BT_PROF(5);
        grid_bar(bar, epoch);
        BT_PROF(6);
        // ================= phase 7: the cut = earliest blocker (or theta); commit before it, undo after it ====
        mkey_t cv = theta; int ci = -1, cp = 0;
        {
            const int nb = (int)min(__ldcg(&g->n_block[rot]), (unsigned)BT_PMAX);
            for (int q = lane; q < nb; q += 32) {
                const BatchBlock b = a.blocks[q];
                if (bt_before(b.ev, b.ei, b.pos, cv, ci, cp)) { cv = b.ev; ci = b.ei; cp = b.pos; }
            }
            // warp reduction of the earliest triple
            for (int o = 16; o > 0; o >>= 1) {
                const mkey_t ov = __shfl_xor_sync(0xffffffffu, cv, o);
                const int oi = __shfl_xor_sync(0xffffffffu, ci, o), op = __shfl_xor_sync(0xffffffffu, cp, o);
                if (bt_before(ov, oi, op, cv, ci, cp)) { cv = ov; ci = oi; cp = op; }
            }
            nblockers += nb;
        }
        for (int r = gwarp; r < n_seeds; r += nwarps) {
            if (sh_label[r] != r) continue;
            const int np = a.npos[r];
            int keep = 0;
            for (int p = 0; p < np; ++p) {
                const BatchElem e = a.elems[(int64_t)r * BT_LMAX + p];
                if (bt_before(e.ev, e.ei, p, cv, ci, cp)) keep = p + 1;        // effective keys never increase along p
            }
            for (int p = np - 1; p >= keep; --p) {                               // undo in reverse order
                const BatchUndo* und = a.undo + ((int64_t)r * BT_LMAX + p) * (Kp + 1);
                const int k = a.elems[(int64_t)r * BT_LMAX + p].k;
                for (int t = lane; t <= Kp; t += 32) {
                    const BatchUndo u = und[t];
                    if (u.idx >= 0) { a.M[u.idx] = u.M; if (t != Kp) a.hdip[u.idx] = u.hd; }
                }
                if (lane == 0) a.s[k] = (int8_t)(-__ldcg(a.s + k));
                __syncwarp();
            }
            for (int p = 0; p < keep; ++p) {                                     // spins the committed flips made switchable
                const BatchUndo* und = a.undo + ((int64_t)r * BT_LMAX + p) * (Kp + 1);
                for (int t = lane; t <= Kp; t += 32) {
                    const int idx = und[t].idx;
                    if (idx >= 0 && __ldcg(a.M + idx) > 1.0) {
                        const unsigned bit = 1u << (idx & 31);
                        if (!(atomicOr(a.cbits + (idx >> 5), bit) & bit)) a.cand[atomicAdd(&g->n_list, 1u)] = idx;
                    }
                }
            }
            if (keep) {
                unsigned base = 0;
                if (lane == 0) base = atomicAdd(&g->n_commit[rot], (unsigned)keep);
                base = __shfl_sync(0xffffffffu, base, 0);
                for (int p = lane; p < keep; p += 32) {
                    const BatchElem e = a.elems[(int64_t)r * BT_LMAX + p];
                    a.clist[base + p] = BatchCommit{~e.ev, ((unsigned long long)(unsigned)e.ei << 32) | (unsigned)p, e.k, 0};
                    if (a.cellidx) a.sgrid[a.cellidx[e.k]] = (__ldcg(a.s + e.k) > 0 ? SG_UP : SG_DOWN);
                }
            }
            if (lane == 0) undone += np - keep;
        }
        grid_bar(bar, epoch);
        BT_PROF(7);
        // ================= phase 8: merged order -> flip log =================================================
        const int nc = (int)__ldcg(&g->n_commit[rot]);
        const long long logbase = nflips % a.log_cap;                             // ring buffer, like k_relax (nc < log_cap)
        for (int q = gwarp; q < nc; q += nwarps) {
            const BatchCommit me = a.clist[q];
            int rank = 0;
            for (int j = lane; j < nc; j += 32) {
                const BatchCommit o = a.clist[j];
                rank += (o.nev < me.nev || (o.nev == me.nev && o.lo < me.lo)) ? 1 : 0;
            }
            rank = __reduce_add_sync(0xffffffffu, rank);
            if (lane == 0) { long long lp = logbase + rank; if (lp >= a.log_cap) lp -= a.log_cap; a.flog[lp] = me.k; }
        }
        BT_PROF(8);
        nflips += nc;
        any_flip |= nc > 0;
        rot = (rot + 1) & 3;
        // a round costs about as much as a few dozen sequential flips: when avalanches are dominoes (every flip
        // triggers the next one) the prefixes stay short and the one-flip-at-a-time loop is faster
        lean = nc < a.min_commit ? lean + 1 : 0;
        if (lean >= 4) { ++rounds; break; }
        // (no barrier: the next round's first pass only reads M, which phase 7 finished before the last barrier;
        //  clist is rewritten only after three more barriers)
    }
    // ================= tail: leaf maxima for k_relax, counters ===============================================
    grid_bar(bar, epoch);
    if (any_flip) {
        const int LB = 1 << a.LBshift;
        for (int b = gwarp; b < a.nblk; b += nwarps) {
            mkey_t bv = 0ull; int bi = 0x7fffffff;
            for (int q = lane; q < LB; q += 32) {
                const int64_t i = ((int64_t)b << a.LBshift) + q;
                if (i < N) {
                    const mkey_t kv = margin_key(__ldcg(a.M + i));
                    if (kv > bv) { bv = kv; bi = (int)i; }
                }
            }
            warp_argmax_key(bv, bi);
            if (lane == 0) {
                a.bval[b] = bv ? __longlong_as_double((long long)bv) : -CUDART_INF;
                a.bidx[b] = bv ? bi : (int)min((int64_t)b << a.LBshift, N - 1);
            }
        }
    }
    // per-warp statistics -> one atomic per warp
    undone = __reduce_add_sync(0xffffffffu, (unsigned)undone);
    if (lane == 0 && undone) atomicAdd((unsigned long long*)&g->undone, (unsigned long long)undone);
    if (blockIdx.x == 0) {                              // leave the control block clean for the next launch
        for (int b = tid; b < 3 * BT_NB; b += BT_THREADS) (&g->hist[0][0])[b] = 0;
        if (tid < 4) { g->n_seeds[tid] = 0; g->n_commit[tid] = 0; g->n_block[tid] = 0; }
        if (tid < 3) g->n_cand[tid] = 0;
        if (tid == 0) { g->bar[parity ^ 1u] = 0; g->launch = g->launch + 1; g->round_base = round_base + (unsigned)rounds; }
    }
    if (gtid == 0) {
        g->flips = nflips; g->rounds = rounds; g->blockers = nblockers;
        a.ctr[0].batch_flips = nflips;
        a.ctr[0].batch_rounds += rounds;
        a.ctr[0].batch_total += nflips;
    }
}
