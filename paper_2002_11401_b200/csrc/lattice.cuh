// lattice.cuh -- regular-lattice detection and the per-sublattice stencil gather (SURVEY.md A2/A3,
// "stencil variant"; BASELINE.json north_star (a): "a per-sublattice stencil for regular lattices so
// g_ij is computed on the fly instead of streamed from HBM").  Included by flatspin.cu only.
//
// On a regular lattice (every flatspin geometry is a Bravais lattice with a basis of
// "sublattices", :146) the coupling alpha*g_ij of Eq. 3 depends only on
// (sublattice of i, sublattice of j, integer cell offset), so the full gather
//     h_dip,i = sum_j s_j alpha g_ij
// is a 2-D correlation of dense per-sublattice spin grids with a table T[sub_i][sub_j][du][dv] of a
// few KB that lives in shared memory: no per-interaction HBM traffic at all.
//
// Nothing is assumed about the input: the lattice is *detected* from raw pos/angle, the table is
// filled from the ELL couplings already computed from the actual positions (k_weights), and the
// result is accepted only if (i) every ELL entry equals its table entry to <= 5e-13/K relative to max|w| and
// (ii) the stencil reaches exactly the ELL's interactions.  Otherwise the ELL gather is used.
//
//   k_lat_assign        sublattice + integer cell of every spin, one pass per sublattice
//   k_lat_extent        bounding box of the cells, stencil half-extents, max |w|
//   k_lat_scatter       dense index grids gidx[sub][v][u] (-1 = empty / halo)
//   k_stencil_owner/fill/verify/rows/count   table construction and the two acceptance checks
//   k_gather_stencil    A3: register-tiled fp64 correlation, FP64-pipe bound
//   k_dfma_peak         DFMA-chain calibration of the FP64 roofline denominator
#pragma once

constexpr int NSUB_MAX = 8;            // more sublattices than this: use the ELL gather
constexpr int STENCIL_RMAX = 40;       // larger stencil half-extent: use the ELL gather
constexpr int ST_OV = 8;               // default outputs per thread along v (sliding register window); 16 is the other variant
constexpr int ST_TU = 32;              // tile extent along u = one warp
// one spin-grid cell = the high word of the spin as a double (+1.0, -1.0, or 0 = no magnet): a 4-byte
// shared-memory load lands directly in the upper register of a DFMA operand whose lower register stays 0
typedef uint32_t sgcell_t;
constexpr sgcell_t SG_UP = 0x3ff00000u, SG_DOWN = 0xbff00000u;

struct LatFrame { double ox, oy, i11, i12, i21, i22; };   // (u, v) = Ainv (r - o)

struct LatGrid {
    int nsub, u0, v0, U, V, Ru, Rv, Up, Vp, W, H;         // W = 2Ru+1, H = 2Rv+1, Up = U+2Ru, Vp = V+2Rv
    int Upa, Vpa;                                         // spin-grid allocation [Vpa][Upa] (u fastest): whole tiles + halo, Upa % 4 == 0
    unsigned inv_nsub;                                    // ceil(2^32 / nsub): z / nsub == umulhi(z, inv_nsub) for z < 2^16, without a division
};

__device__ __forceinline__ void lat_uv(const LatFrame& f, double2 p, double& u, double& v) {
    double x = p.x - f.ox, y = p.y - f.oy;
    u = f.i11 * x + f.i12 * y;
    v = f.i21 * x + f.i22 * y;
}

// One pass per sublattice: every still-unassigned spin with the representative's orientation whose
// lattice coordinates differ from the representative's by integers joins sublattice `pass`.
// next[0] = lowest index still unassigned after this pass; next[1] += assigned.
__global__ void k_lat_assign(int64_t N, LatFrame f, int rep, int pass, const double2* __restrict__ pos,
                             const double2* __restrict__ cs, uint8_t* __restrict__ sub, int* __restrict__ cu,
                             int* __restrict__ cv, int* __restrict__ next) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    bool took = false, left = false;
    if (i < N && sub[i] == 0xff) {
        double u, v, ur, vr;
        lat_uv(f, pos[i], u, v);
        lat_uv(f, pos[rep], ur, vr);
        double2 c = cs[i], cr = cs[rep];
        double du = u - ur, dv = v - vr, ru = rint(du), rv = rint(dv);
        bool same = fabs(c.x - cr.x) < 1e-9 && fabs(c.y - cr.y) < 1e-9;
        if (same && fabs(du - ru) < 1e-6 && fabs(dv - rv) < 1e-6 && fabs(ru) < 1e9 && fabs(rv) < 1e9) {
            sub[i] = (uint8_t)pass;
            cu[i] = (int)ru + (int)rint(ur);
            cv[i] = (int)rv + (int)rint(vr);
            took = true;
        } else {
            left = true;
        }
    }
    unsigned mt = __ballot_sync(0xffffffffu, took), ml = __ballot_sync(0xffffffffu, left);
    if ((threadIdx.x & 31) == 0) {
        if (mt) atomicAdd(&next[1], __popc(mt));
        if (ml) atomicMin(&next[0], (int)(i - (threadIdx.x & 31)) + (__ffs(ml) - 1));
    }
}

// ext[0..3] = min cu, min cv, max cu, max cv; ext[4], ext[5] = max |du|, |dv| over ELL entries;
// wmax = bits of max |w| (positive doubles order like their bit patterns).
__global__ void k_lat_extent(int64_t N, int Kp, const int* __restrict__ nbr, const double2* __restrict__ w,
                             const int* __restrict__ cu, const int* __restrict__ cv, int* __restrict__ ext,
                             unsigned long long* __restrict__ wmax) {
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int ru = 0, rv = 0, ulo = 0x7fffffff, vlo = 0x7fffffff, uhi = (int)0x80000000, vhi = (int)0x80000000;
    double wm = 0.0;
    if (t < N * Kp) {
        int64_t i = t / Kp;
        int j = nbr[t];
        int ui = cu[i], vi = cv[i];
        if (j >= 0) {
            ru = abs(cu[j] - ui); rv = abs(cv[j] - vi);
            double2 ww = w[t];
            wm = fmax(fabs(ww.x), fabs(ww.y));
        }
        ulo = uhi = ui; vlo = vhi = vi;
    }
    // one set of atomics per warp, and only if it can change the result (plain reads first)
    ru = __reduce_max_sync(0xffffffffu, ru); rv = __reduce_max_sync(0xffffffffu, rv);
    ulo = __reduce_min_sync(0xffffffffu, ulo); vlo = __reduce_min_sync(0xffffffffu, vlo);
    uhi = __reduce_max_sync(0xffffffffu, uhi); vhi = __reduce_max_sync(0xffffffffu, vhi);
    for (int o = 16; o > 0; o >>= 1) wm = fmax(wm, __shfl_xor_sync(0xffffffffu, wm, o));
    if ((threadIdx.x & 31) == 0) {
        volatile int* e = ext;
        if (ulo < e[0]) atomicMin(&ext[0], ulo);
        if (vlo < e[1]) atomicMin(&ext[1], vlo);
        if (uhi > e[2]) atomicMax(&ext[2], uhi);
        if (vhi > e[3]) atomicMax(&ext[3], vhi);
        if (ru > e[4]) atomicMax(&ext[4], ru);
        if (rv > e[5]) atomicMax(&ext[5], rv);
        unsigned long long wb = (unsigned long long)__double_as_longlong(wm);
        if (wb > *(volatile unsigned long long*)wmax) atomicMax(wmax, wb);
    }
}

__device__ __forceinline__ int64_t lat_cell(const LatGrid& g, int sub, int cu, int cv) {
    return ((int64_t)sub * g.Vp + (cv - g.v0 + g.Rv)) * g.Up + (cu - g.u0 + g.Ru);
}

// flags bit 2: two spins in one cell.  cellidx[i] = position of spin i in one replica's spin grid sg[sub][Vpa][Upa].
__global__ void k_lat_scatter(int64_t N, LatGrid g, const uint8_t* __restrict__ sub, const int* __restrict__ cu,
                              const int* __restrict__ cv, int* __restrict__ gidx, int* __restrict__ cellidx,
                              int* __restrict__ flags) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    cellidx[i] = (int)(((int64_t)sub[i] * g.Vpa + (cv[i] - g.v0 + g.Rv)) * g.Upa + (cu[i] - g.u0 + g.Ru));
    if (atomicCAS(&gidx[lat_cell(g, sub[i], cu[i], cv[i])], -1, (int)i) != -1) atomicOr(flags, 4);
}

__device__ __forceinline__ int64_t stencil_slot(const LatGrid& g, int si, int sj, int du, int dv) {
    return ((int64_t)(si * g.nsub + sj) * g.W + (du + g.Ru)) * g.H + (dv + g.Rv);
}

// mode 0: owner[slot] = lowest ELL entry that maps to it; mode 1: the owner writes T[slot];
// mode 2: dev = bits of max |w - T| over all entries.
__global__ void k_stencil_build(int mode, int64_t N, int Kp, LatGrid g, const int* __restrict__ nbr,
                                const double2* __restrict__ w, const uint8_t* __restrict__ sub,
                                const int* __restrict__ cu, const int* __restrict__ cv,
                                unsigned long long* __restrict__ owner, double2* __restrict__ T,
                                unsigned long long* __restrict__ dev) {
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double d = 0.0;
    if (t < N * Kp) {
        int64_t i = t / Kp;
        int j = nbr[t];
        if (j >= 0) {
            int64_t slot = stencil_slot(g, sub[i], sub[j], cu[j] - cu[i], cv[j] - cv[i]);
            if (mode == 0) { if (*(volatile unsigned long long*)(owner + slot) > (unsigned long long)t) atomicMin(&owner[slot], (unsigned long long)t); }
            else if (mode == 1) { if (owner[slot] == (unsigned long long)t) T[slot] = w[t]; }
            else { double2 a = w[t], b = T[slot]; d = fmax(fabs(a.x - b.x), fabs(a.y - b.y)); }
        }
    }
    if (mode == 2) {
        for (int o = 16; o > 0; o >>= 1) d = fmax(d, __shfl_xor_sync(0xffffffffu, d, o));
        if ((threadIdx.x & 31) == 0 && d > 0.0 && (unsigned long long)__double_as_longlong(d) > *(volatile unsigned long long*)dev)
            atomicMax(dev, (unsigned long long)__double_as_longlong(d));
    }
}

// rowtab[(pair * W + du)] = (dvmin, dvmax) of the present slots of that row, (1, 0) if the row is empty
__global__ void k_stencil_rows(LatGrid g, const unsigned long long* __restrict__ owner, int2* __restrict__ rowtab) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.nsub * g.nsub * g.W) return;
    const unsigned long long* o = owner + (int64_t)t * g.H;
    int lo = 1, hi = 0;
    bool any = false;
    for (int k = 0; k < g.H; ++k)
        if (o[k] != ~0ull) { if (!any) lo = k - g.Rv; hi = k - g.Rv; any = true; }
    rowtab[t] = any ? make_int2(lo, hi) : make_int2(1, 0);
}

// acceptance check (ii): number of (spin, present slot, occupied cell) triples == number of ELL entries
__global__ void k_stencil_count(int64_t N, LatGrid g, const uint8_t* __restrict__ sub, const int* __restrict__ cu,
                                const int* __restrict__ cv, const int* __restrict__ gidx,
                                const unsigned long long* __restrict__ owner, unsigned long long* __restrict__ total) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    unsigned long long n = 0;
    if (i < N) {
        int si = sub[i], ui = cu[i], vi = cv[i];
        for (int sj = 0; sj < g.nsub; ++sj)
            for (int du = -g.Ru; du <= g.Ru; ++du)
                for (int dv = -g.Rv; dv <= g.Rv; ++dv)
                    if (owner[stencil_slot(g, si, sj, du, dv)] != ~0ull && gidx[lat_cell(g, sj, ui + du, vi + dv)] >= 0) ++n;
    }
    for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(total, n);
}

// dense spin grids sg[rep][sub][Vpa][Upa] (u fastest, like gidx), one sgcell_t per lattice site, rebuilt from s when
// the spins were rewritten from outside (the relax loop keeps them in step with its own flips).
__global__ void k_spin_grid(int64_t N, LatGrid g, int R, const int* __restrict__ gidx, const int8_t* __restrict__ s_all,
                            sgcell_t* __restrict__ sg) {
    const int sub = blockIdx.z;
    const int gu = blockIdx.x * 32 + (threadIdx.x & 31);
    for (int gv = blockIdx.y * 32 + (threadIdx.x >> 5); gv < min(g.Vp, (int)(blockIdx.y + 1) * 32); gv += 8) {
        if (gu >= g.Up) continue;
        const int idx = gidx[((int64_t)sub * g.Vp + gv) * g.Up + gu];
        for (int r = 0; r < R; ++r) {
            const int sv = idx >= 0 ? (int)s_all[(int64_t)r * N + idx] : 0;
            sg[(((int64_t)r * g.nsub + sub) * g.Vpa + gv) * g.Upa + gu] = (sv > 0 ? SG_UP : (sv < 0 ? SG_DOWN : 0u));
        }
    }
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// TMA (cp.async.bulk.tensor) + mbarrier, used by the inversion-paired fp64 kernel for its spin tiles: one thread issues
// one 3-D box copy per source sublattice (box = PU cells x SH rows x 1 grid; cells outside the grid arrive as zeros).
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_%=;\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2),
                   "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

// ------------------------------------------------------------------------------------------------
// A3, stencil variant.  CTA = NW x RS warps; tile = 32 cells along u (one per lane) x 8*NW cells
// along v (8 consecutive outputs per thread).  Prologue: the spin tiles (+ halo, 4-byte cells) of every
// source sublattice, the row intervals and the spin index of every output go to shared memory with
// cp.async in one shot (one global round trip per CTA, no staging through registers).  Main loop: for
// each stencil row du the thread slides an 8-wide register window along v, which is the contiguous
// direction of its shared-memory row (immediate offsets, odd row pitch so the 32 lanes hit 32 banks);
// per stencil slot one 4-byte shared load (the high word of a double whose low word is zero) and the
// weight pair (CT variant: two uniform-register loads through the constant cache; otherwise one
// broadcast 16-byte shared load) feed 16 DFMA.  The stencil rows are dealt round-robin to RS warp
// groups that share the tile (RS times the warps for the same shared-memory traffic: the FP64 pipe
// wants >= 4 warps per scheduler); their partial sums are added through shared memory in a fixed order.
// blockIdx.z = replica * nsub + target sublattice.  blockDim = 32 * NW * RS.
// ------------------------------------------------------------------------------------------------
// Coupling tables of the lattice that used the stencil last (all sublattice pairs), for the CT variant of
// k_gather_stencil: a warp-uniform weight read through the constant cache lands in a uniform register,
// and DFMA R, R, UR, R reads only two vector-register pairs: 62 DFMA/clk/SM measured against 51 with
// the weight in a vector register.  Re-uploaded when another simulation takes over.
constexpr int CT_MAX = 2560;           // double2 entries (40 KB of the 64 KB constant bank)
constexpr int CR_MAX = 960;            // row intervals (7.5 KB)
constexpr int CP_MAX = 480;            // row pairs of the inversion-symmetric variant (7.5 KB)
__constant__ double2 c_T[CT_MAX];
__constant__ int2 c_rows[CR_MAX];
// Inversion symmetry (Eq. 3, is even in r_ij): T[si][sj][du][dv] == T[si][sj][-du-cu][-dv-cv] for the
// lattice's inversion offset (cu, cv) of that sublattice pair.  The SYM variant visits only one slot of every such
// pair: x(+d) + x(-d) once (DADD), then one DFMA pair: 3 FP64 operations per 2 interactions instead of 4.
// c_prow[e] = {row+ | row- << 16, first dv of row+, last dv of row+, offset of the mirrored window in row-};
// c_pstart[pair] = {first entry, entries}.
__constant__ int4 c_prow[CP_MAX];
__constant__ int2 c_pstart[NSUB_MAX * NSUB_MAX];
// Table offset of the first slot of every row (plain) / row pair (SYM), in arrays of their own: a value whose only
// consumer is the index of c_T stays in the uniform datapath (LDCU -> UR -> LDCU.64 c_T[UR + imm] -> DFMA R, R, UR, R);
// derived from a row entry that also feeds vector address arithmetic, ptxas loads it into a vector register and the
// weights follow (LDC.64, DFMA with three vector operands: 51 instead of 62 DFMA/clk/SM).
__constant__ int c_rtofs[CR_MAX];
__constant__ CUtensorMap c_sg_map;     // TMA descriptor of the owner's spin grids (uploaded with the tables)
__constant__ int c_ptofs[CP_MAX];

// scalar helpers of the stencil kernel: R = double (the parity path) or float (the optional fp32 field path of
// BASELINE.json north_star, reported separately at 1e-5; it converts the spin cells while staging them and reads a
// float2 copy of the table through the same constant array)
template <typename R> __device__ __forceinline__ R st_cell(sgcell_t c);
template <> __device__ __forceinline__ double st_cell<double>(sgcell_t c) { return __hiloint2double((int)c, 0); }
template <> __device__ __forceinline__ float st_cell<float>(sgcell_t c) { return __uint_as_float(c); }
template <typename R> struct StPair { R x, y; };
template <typename R> __device__ __forceinline__ StPair<R> ct_load(int i);
template <> __device__ __forceinline__ StPair<double> ct_load<double>(int i) { const double2 t = c_T[i]; return StPair<double>{t.x, t.y}; }
template <> __device__ __forceinline__ StPair<float> ct_load<float>(int i) {
    const float2 t = reinterpret_cast<const float2*>(c_T)[i]; return StPair<float>{t.x, t.y};
}
__device__ __forceinline__ double st_fma(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float st_fma(float a, float b, float c) { return fmaf(a, b, c); }
// the high word of +-1.0 / 0 as a double -> the bits of +-1.0f / 0
__device__ __forceinline__ unsigned cell_to_f32(unsigned c) { return (c & 0x80000000u) | (c ? 0x3f800000u : 0u); }

template <int MAXT, int MINB, bool CT, int OV, bool SYM, int PU, typename R = double>
__global__ void __launch_bounds__(MAXT, MINB) k_gather_stencil(int64_t N, LatGrid g, int NW, int Pv,
                                                               const int* __restrict__ gidx, const sgcell_t* __restrict__ sg,
                                                               const double2* __restrict__ T, const int2* __restrict__ rowtab,
                                                               double2* __restrict__ hdip_all) {
    asm volatile("griddepcontrol.launch_dependents;");   // lets a following k_scan become resident in this kernel's tail (see k_scan)
    extern __shared__ __align__(128) unsigned char st_raw[];
    const int RS = (blockDim.x >> 5) / NW, TV = OV * NW;
    const int SUc = (ST_TU + 2 * g.Ru + 3) & ~3, SH = TV + 2 * g.Rv, WH = g.W * g.H;   // staged row: SUc cells, pitch PU
    (void)Pv;
    constexpr bool F32 = sizeof(R) == 4;
    static_assert(!F32 || CT, "the fp32 variant reads its table from constant memory");
    double2* Tsm = reinterpret_cast<double2*>(st_raw);                      // [nsub][WH]
    const size_t tsm_n = CT ? 0 : (size_t)g.nsub * WH;                      // no shared copy of T in the CT variant
    int2* rows = reinterpret_cast<int2*>(Tsm + tsm_n);                      // [nsub][W]
    int* oidx = reinterpret_cast<int*>(rows + (size_t)g.nsub * g.W);        // [TV][32] spin index of every output
    sgcell_t* S = reinterpret_cast<sgcell_t*>(st_raw + ((16 * tsm_n + 8 * (size_t)g.nsub * g.W + 128 * TV + 8 + 127) & ~(size_t)127));   // [nsub][SH][PU], 128-byte aligned (TMA)
    constexpr bool TMA = SYM && CT && sizeof(R) == 8;                       // the headline variant stages its tiles by TMA
    // No division: ptxas computes one in the vector datapath and, in some instantiations (fp32, 256-thread CTAs), then kept
    // si, the row tables indexed with it and finally the weights in vector registers (LDC + three-vector-operand DFMA).
    const int rep = g.nsub == 1 ? (int)blockIdx.z : (int)__umulhi(blockIdx.z, g.inv_nsub), si = (int)blockIdx.z - rep * g.nsub;
    const int tu0 = blockIdx.x * ST_TU, tv0 = blockIdx.y * TV;       // tile origin, interior coordinates
    // the warp index via a shuffle from lane 0: the compiler then knows everything derived from it is
    // warp-uniform
    const int wid_u = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31, warp = wid_u % NW, rs = wid_u / NW;

    // (the mbarrier of the TMA variant: the last 8 bytes in front of the tiles, inside the 128-byte alignment pad)
    unsigned long long* tma_bar = reinterpret_cast<unsigned long long*>(S) - 1;
    (void)tma_bar;
    // ---- prologue: everything this CTA reads, in flight at once.  A staged row = SUc consecutive cells along u
    // (contiguous in the spin grid and in shared memory): 16-byte cp.async, 16 or 32 lanes per row
    {
        const sgcell_t* src = sg + (((int64_t)rep * g.nsub * g.Vpa + tv0) * g.Upa + tu0);
        constexpr int CPR = PU / 4;                                   // 16-byte chunks per shared-memory row
        const int nch = SUc >> 2;
        // a thread keeps its chunk column and walks down the rows with constant strides (the generic (row, chunk) = t / CPR,
        // t % CPR loop with 64-bit addresses cost ~25 instructions per copy: 6% of the kernel's instructions)
        if constexpr (TMA) {
            // one thread: barrier, expected bytes, one box copy per source sublattice (coordinates in the padded spin grid;
            // a box is PU cells wide: what lies beyond the grid arrives as zeros).  Everybody waits on the barrier below.
            // (no loop inside a divergent branch, here or below: behind one, ptxas no longer treats the main loop as
            // convergent and moves its weights out of the uniform datapath)
            if (threadIdx.x == 0) mbar_init(tma_bar, 1);
            __syncthreads();                                          // the initialised barrier is visible to every thread
            if (threadIdx.x == 0) mbar_expect_tx(tma_bar, (unsigned)(g.nsub * SH * PU * (int)sizeof(sgcell_t)));
            for (int sj = 0; sj < g.nsub; ++sj)
                if (threadIdx.x == 0) tma_load_3d(S + (size_t)sj * SH * PU, &c_sg_map, tu0, tv0, rep * g.nsub + sj, tma_bar);
        } else if constexpr (F32) {                                   // staged through registers: cells become float bits
            for (int sj = 0; sj < g.nsub; ++sj) {
                sgcell_t* dst = S + (size_t)sj * SH * PU;
                const sgcell_t* srcj = src + (int64_t)sj * g.Vpa * g.Upa;
                for (int t = threadIdx.x; t < SH * CPR; t += blockDim.x) {
                    const int vl = t / CPR, ch = t % CPR;             // CPR is a power of two
                    if (ch < nch) {
                        uint4 v = __ldg(reinterpret_cast<const uint4*>(srcj + (int64_t)vl * g.Upa + 4 * ch));
                        v.x = cell_to_f32(v.x); v.y = cell_to_f32(v.y); v.z = cell_to_f32(v.z); v.w = cell_to_f32(v.w);
                        *reinterpret_cast<uint4*>(dst + (size_t)vl * PU + 4 * ch) = v;
                    }
                }
            }
        } else {
            const int ch = threadIdx.x & (CPR - 1), vl0 = threadIdx.x / CPR, vstep = blockDim.x / CPR;
            const bool mine = ch < nch;                               // (the loops themselves stay free of divergent branches)
            for (int sj = 0; sj < g.nsub; ++sj) {
                sgcell_t* d = S + ((size_t)sj * SH + vl0) * PU + 4 * ch;
                const sgcell_t* p = src + ((int64_t)sj * g.Vpa + vl0) * g.Upa + 4 * ch;
                const int64_t pstep = (int64_t)vstep * g.Upa;
#pragma unroll 4
                for (int vl = vl0; vl < SH; vl += vstep, d += vstep * PU, p += pstep)
                    if (mine) cp_async16(d, p);
            }
        }
    }
    if (!CT)
        for (int t = threadIdx.x; t < g.nsub * WH; t += blockDim.x) cp_async16(Tsm + t, T + (int64_t)si * g.nsub * WH + t);
    if (!CT)
        for (int t = threadIdx.x; t < g.nsub * g.W; t += blockDim.x) rows[t] = __ldg(rowtab + si * g.nsub * g.W + t);
    for (int t = threadIdx.x; t < TV * 32; t += blockDim.x) {
        int gu = tu0 + (t & 31) + g.Ru, gv = tv0 + (t >> 5) + g.Rv;
        if (gu < g.Up && gv < g.Vp) cp_async4(oidx + t, gidx + ((int64_t)si * g.Vp + gv) * g.Up + gu);
        else oidx[t] = -1;
    }
    cp_async_wait_all();
    if constexpr (TMA) mbar_wait(tma_bar, 0);           // every thread observes the completion of the box copies itself
    __syncthreads();

    R ax[OV], ay[OV], x[OV];                           // all indices below are compile-time after unrolling: registers
#pragma unroll
    for (int q = 0; q < OV; ++q) { ax[q] = (R)0; ay[q] = (R)0; }
#define FS_ST_LD(K) st_cell<R>(sp[(K) * PU])
#define FS_ST_LDM(K) st_cell<R>(sm[(K) * PU])

    if (SYM) {
        // one slot of every inversion pair: window x slides forward along row+, window y backward along row-
        R y[OV];
        for (int sj = 0; sj < g.nsub; ++sj) {
            const sgcell_t* Sj = S + ((size_t)sj * SH + warp * OV + g.Rv) * PU + lane;
            const int2 ps = c_pstart[si * g.nsub + sj];
            for (int e = 0; e < ps.y; ++e) {
                if ((e & (RS - 1)) != rs) continue;
                const int4 pr = c_prow[ps.x + e];
                const int rp = pr.x & 0xffff, rm = pr.x >> 16;
                int n = pr.z - pr.y + 1;
                const sgcell_t* sp = Sj + rp + pr.y * PU;              // x[q] = S[.. + q + dv][lane + row+]
                const sgcell_t* sm = Sj + rm + pr.w * PU;              // y[q] = S[.. + q - dv - cv][lane + row-]
                int tofs = c_ptofs[ps.x + e];
#pragma unroll
                for (int q = 0; q < OV; ++q) { x[q] = FS_ST_LD(q); y[q] = FS_ST_LDM(q); }
                for (; n >= OV; n -= OV, sp += OV * PU, sm -= OV * PU, tofs += OV) {
#pragma unroll
                    for (int K = 0; K < OV; ++K) {
                        const StPair<R> t = ct_load<R>(tofs + K);
#pragma unroll
                        for (int q = 0; q < OV; ++q) {
                            const R z = x[(q + K) % OV] + y[(q - K + OV) % OV];
                            ax[q] = st_fma(z, t.x, ax[q]);
                            ay[q] = st_fma(z, t.y, ay[q]);
                        }
                        x[K] = FS_ST_LD(OV + K);
                        y[OV - 1 - K] = FS_ST_LDM(-(K + 1));
                    }
                }
                if (n > 0) {
#pragma unroll
                    for (int K = 0; K < OV - 1; ++K) {
                        const StPair<R> t = ct_load<R>(tofs + K);
#pragma unroll
                        for (int q = 0; q < OV; ++q) {
                            const R z = x[(q + K) % OV] + y[(q - K + OV) % OV];
                            ax[q] = st_fma(z, t.x, ax[q]);
                            ay[q] = st_fma(z, t.y, ay[q]);
                        }
                        if (--n == 0) break;
                        x[K] = FS_ST_LD(OV + K);
                        y[OV - 1 - K] = FS_ST_LDM(-(K + 1));
                    }
                }
            }
        }
    } else
    for (int sj = 0; sj < g.nsub; ++sj) {
        const sgcell_t* Sj = S + ((size_t)sj * SH + warp * OV + g.Rv) * PU + lane;
        const double2* Tj = Tsm + (CT ? 0 : (size_t)sj * WH + g.Rv);
        const int tj = (si * g.nsub + sj) * WH + g.Rv;
        // r = du + Ru is a uniform loop counter, so that the row interval and the weight offsets below live
        // in uniform registers (starting every CTA at a different row to break lockstep was tried: no gain)
        for (int r = 0; r < g.W; ++r) {
            if ((r & (RS - 1)) != rs) continue;        // RS is a power of two
            const int2 rt = CT ? c_rows[(si * g.nsub + sj) * g.W + r] : rows[sj * g.W + r];
            int n = rt.y - rt.x + 1;
            if (n <= 0) continue;
            // output (lane, warp*OV+q) at slot (du, dv) reads S[sj][warp*OV + q + dv + Rv][lane + du + Ru]
            const sgcell_t* sp = Sj + r + rt.x * PU;
            const double2* tp = Tj + (CT ? 0 : r * g.H + rt.x);
            int tofs = CT ? c_rtofs[(si * g.nsub + sj) * g.W + r] : tj + r * g.H + rt.x;
#pragma unroll
            for (int q = 0; q < OV; ++q) x[q] = FS_ST_LD(q);
            // full groups of OV slots (no exit test): slot K consumes the window and refills its oldest cell
            for (; n >= OV; n -= OV, sp += OV * PU, tp += OV, tofs += OV) {
#pragma unroll
                for (int K = 0; K < OV; ++K) {
                    StPair<R> t;
                    if (CT) t = ct_load<R>(tofs + K); else { const double2 tt = tp[K]; t = StPair<R>{(R)tt.x, (R)tt.y}; }
#pragma unroll
                    for (int q = 0; q < OV; ++q) {
                        ax[q] = st_fma(x[(q + K) % OV], t.x, ax[q]);
                        ay[q] = st_fma(x[(q + K) % OV], t.y, ay[q]);
                    }
                    x[K] = FS_ST_LD(OV + K);
                }
            }
            if (n > 0) {                               // ragged tail: at most OV - 1 slots
#pragma unroll
                for (int K = 0; K < OV - 1; ++K) {
                    StPair<R> t;
                    if (CT) t = ct_load<R>(tofs + K); else { const double2 tt = tp[K]; t = StPair<R>{(R)tt.x, (R)tt.y}; }
#pragma unroll
                    for (int q = 0; q < OV; ++q) {
                        ax[q] = st_fma(x[(q + K) % OV], t.x, ax[q]);
                        ay[q] = st_fma(x[(q + K) % OV], t.y, ay[q]);
                    }
                    if (--n == 0) break;
                    x[K] = FS_ST_LD(OV + K);
                }
            }
        }
    }
#undef FS_ST_LD
#undef FS_ST_LDM
    // ---- epilogue: add the row groups' partial sums (fixed order), scatter the OV outputs to their spins
    if (RS > 1) {
        __syncthreads();                               // everyone is done with the tiles
        R* red_base = reinterpret_cast<R*>(S);
        R* red = red_base + ((size_t)((rs - 1) * NW + warp) * 2 * OV) * 32 + lane;
        if (rs > 0) {
#pragma unroll
            for (int q = 0; q < OV; ++q) { red[(2 * q) * 32] = ax[q]; red[(2 * q + 1) * 32] = ay[q]; }
        }
        __syncthreads();
        if (rs > 0) return;
        for (int k = 1; k < RS; ++k) {
            const R* rd = red_base + ((size_t)((k - 1) * NW + warp) * 2 * OV) * 32 + lane;
#pragma unroll
            for (int q = 0; q < OV; ++q) { ax[q] += rd[(2 * q) * 32]; ay[q] += rd[(2 * q + 1) * 32]; }
        }
    }
    double2* __restrict__ hdip = hdip_all + (int64_t)rep * N;
    const int* oi = oidx + (warp * OV) * 32 + lane;
#pragma unroll
    for (int q = 0; q < OV; ++q) {
        const int i = oi[q * 32];
        if (i >= 0) hdip[i] = make_double2((double)ax[q], (double)ay[q]);
    }
}

__global__ void k_table_f32(int n, const double2* __restrict__ T, float2* __restrict__ Tf) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) { const double2 v = T[t]; Tf[t] = make_float2((float)v.x, (float)v.y); }
}

// FFMA-chain calibration of the fp32 roofline denominator (the optional fp32 field path)
__global__ void k_ffma_peak(int iters, float seed, float* __restrict__ sink) {
    float a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6, a7 = seed + 7;
    const float m = 1.0000001f, c = 1e-9f * threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < iters; ++k) {
        a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
        a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
    }
    float r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 12345.678f) sink[0] = r;
}

// DFMA-chain calibration: every thread runs 8 independent chains of `iters` DFMAs.
__global__ void k_dfma_peak(int iters, double seed, double* __restrict__ sink) {
    double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6, a7 = seed + 7;
    const double m = 1.0000001, c = 1e-9 * threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < iters; ++k) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    double r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 12345.678) sink[0] = r;                   // never true; keeps the chains alive
}
