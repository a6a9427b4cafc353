// flatspin.cu -- B200 (sm_100a) kernels + C ABI of the flatspin hot path (include/flatspin.h).
//
// Written from /root/reference/PAPER.md (arxiv 2002.11401); PAPER.md lines are cited per kernel.
// Shares no code with oracle/ (the CPU oracle) and never calls it.  No CPU fallback.
//
// Kernels (DESIGN.md "Kernels" has the roofline of each):
//   k_frame            A0  cos/sin tables, hc validation                      (Eq. 1)
//   k_bbox, k_cell_*   A1  cell grid (counting sort)
//   k_count_neighbors  A1  degree of every spin, coincidence check
//   k_fill_neighbors   A1  warp-per-spin collection + bitonic sort -> row-major ELL, ascending
//   k_weights          A2  w_ij = alpha g_ij and its transpose                (Eq. 3)
//   k_gather<G>        A3  h_dip,i = sum_k s_j w_ij, G lanes cooperate per row
//   k_scan             A4-A7 total field + Philox thermal + astroid + margin + leaf-block arg-max
//                                                                             (Eqs. 2,5,6)
//                      (+ top-level arg-max and switchable count by the last CTA to finish, for fs_scan)
//   k_relax            A7-A9 persistent single-CTA-per-replica relax loop with incremental updates
//                                                                             (Eq. 3 linear in s_j)
//   k_fields_out       fs_get_fields
//   lattice.cuh        lattice detection + stencil tables + k_gather_stencil (A3, FP64-bound variant)
#include <cuda.h>                  // CUtensorMap (the driver entry point is fetched at run time: no link against libcuda)
#include <cuda_runtime.h>
#include <math_constants.h>

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <algorithm>
#include <vector>

#include "flatspin.h"

namespace {

// ------------------------------------------------------------------------------------------------
// host-side helpers
// ------------------------------------------------------------------------------------------------
thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};
// ownership of the constant-memory coupling table (lattice.cuh c_T)
std::mutex g_ct_mutex;
unsigned long long g_ct_owner_dev[64] = {0};               // per device: __constant__ memory and events are per device
std::atomic<unsigned long long> g_ct_next_id{0};
cudaEvent_t g_ct_event_dev[64] = {nullptr};

int fail(int code, const char* fmt, ...) {
    va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap);
    return code;
}
#define CUDA_TRY(expr)                                                                             \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail(FS_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
    } while (0)
#define LAUNCHED() (g_launches.fetch_add(1, std::memory_order_relaxed))

constexpr int MAX_LEAF_BLOCKS = 16384;  // leaf-block maxima kept in the relax CTA's shared memory (12 B each + groups: 203 KB of 227):
                                        // leaves of up to 1024 spins, so N <= 16,777,216 spins per replica
constexpr int MAX_K = 8192;             // maximum degree supported by the warp bitonic sort

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// The dynamic shared-memory limit is an attribute of the kernel function (per device), not of a simulation:
// it is only ever raised, so that simulations of different sizes can coexist in one process.
std::mutex g_smem_mutex;
std::map<std::pair<const void*, int>, size_t> g_smem_limit;   // (kernel, device) -> limit set so far
template <typename F>
cudaError_t raise_smem_limit(F* func, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(g_smem_mutex);
    size_t& cur = g_smem_limit[std::make_pair((const void*)func, dev)];
    if (bytes <= cur) return cudaSuccess;
    e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) cur = bytes;
    return e;
}

// Launch with programmatic stream serialisation allowed: the kernel may become resident before the kernel in front of it
// in the stream has finished, if that kernel executed griddepcontrol.launch_dependents; it must execute griddepcontrol.wait
// before it touches anything an earlier kernel writes or reads.  Hides the launch latency of back-to-back dependent kernels.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// every entry point runs on the simulation's device, whatever device is current in the calling thread
struct DeviceGuard {
    int prev = -1, dev;
    explicit DeviceGuard(int d) : dev(d) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; if (prev != dev) cudaSetDevice(dev); }
    ~DeviceGuard() { if (prev >= 0 && prev != dev) cudaSetDevice(prev); }
};

struct Counters {            // one per replica, device resident
    long long total_flips;
    long long last_flips;
    long long n_switchable;
    long long best_index;
    double best_L;
    int status;              // 1 = stopped by max_flips
    int last_step;           // sweep mode: index of the last step reached (T - 1 unless the cap stopped it)
    long long batch_flips;   // flips committed by k_relax_batch in the current relax (k_relax continues from here)
    long long batch_total, batch_rounds;   // since creation / the last reset: flips and rounds of k_relax_batch
    unsigned int ticket;     // k_scan: CTAs of this replica that have finished (last one finalises)
    unsigned long long acc_switch;   // k_scan: running count of switchable spins
};

// ------------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool better(double va, int ia, double vb, int ib) {
    // arg-max key: value descending, index ascending (lowest index wins exact ties; reading C-7)
    return (va > vb) || (va == vb && ia < ib);
}

// Philox4x32-10 (Salmon et al. SC'11), restated for the device.  counter = (spin, step, 0, 0),
// key = (seed_lo, seed_hi)  (reading C-11).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// thermal field of spin i at `step` in global x,y: sigma * (z0, z1), Box-Muller on two 52-bit uniforms
// (reading C-11)
__device__ __forceinline__ double2 thermal_xy(double sigma, uint64_t seed, uint32_t step, uint32_t i) {
    uint32_t x[4];
    philox4x32_10(i, step, 0u, 0u, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32), x);
    // u = (a + 1/2) 2^-52 with a = the top 52 bits: the bits of a are the mantissa of a double in [1, 2), so
    // u = (1.a - 1) + 2^-53, both steps exact (no 64-bit integer-to-double conversion)
    const double half_ulp = 1.0 / 9007199254740992.0;
    const double u1 = (__hiloint2double((int)(0x3ff00000u | (x[0] >> 12)), (int)((x[0] << 20) | (x[1] >> 12))) - 1.0) + half_ulp;
    const double u2 = (__hiloint2double((int)(0x3ff00000u | (x[2] >> 12)), (int)((x[2] << 20) | (x[3] >> 12))) - 1.0) + half_ulp;
    const double r = sqrt(-2.0 * log(u1));
    // cos / sin of 2 pi u2 by sincospi(2 u2): the angle's range reduction is exact and cheap; the result differs from
    // cos(fl(2 pi u2)) by the rounding of that product (<= 7e-16 absolute), like every other few-ulp difference of D-3
    double sn, cs;
    sincospi(2.0 * u2, &sn, &cs);
    return make_double2(sigma * r * cs, sigma * r * sn);
}

struct Astroid {           // 1/b, 1/c, 2/gamma, 2/beta, power kinds; tx, ty: both terms of Eq. 5 below 1/2 (see margin())
    double inv_b, inv_c, e_par, e_perp; int k_par, k_perp; double tx, ty;
};

// x^e for x >= 0, e > 0.  kind 1: e = 2/3 (gamma or beta = 3, the classical astroid, Eq. 4)
// -> cbrt(x^2); kind 2: e = 1; kind 3: e = 2; else exp(e log x).  On this path (one warp, a dependent
// chain per flip) CUDA's pow costs ~770 cycles, exp(log) ~450, cbrt ~310 (measured); all are within a
// few ulp of the exact power, far inside the 1e-12 parity bar and the >= 1e-10 decision gaps (D-3).
__device__ __forceinline__ double pow_kind(double x, double e, int kind) {
    if (kind == 1) return cbrt(x * x);
    if (kind == 2) return x;
    if (kind == 3) return x * x;
    return x > 0.0 ? exp(e * log(x)) : 0.0;
}

// switching margin M_i (Eq. 5 left-hand side if Eq. 6 holds, else -inf): PAPER.md:103, :112.
// ihc = 1 / h_c^(i), precomputed once (k_frame).
__device__ __forceinline__ double margin(double hpar, double hperp, double s, double ihc, const Astroid& a) {
    if (!(s * hpar < 0.0)) return -CUDART_INF;
    double x = fabs(hpar) * (a.inv_b * ihc);
    double y = fabs(hperp) * (a.inv_c * ihc);
    // Well inside the astroid (each term of Eq. 5 below 1/2, with a 1e-9 guard band for the few-ulp powers): the spin cannot
    // switch and cannot be the arg-max that matters (only margins > 1 ever win), so its margin is recorded as 0 ("not
    // switchable", the same key as -inf) and the two fractional powers are skipped.  Whole-protocol scans spend most of
    // their FP64 work on such spins (ensembles of small systems are FP64-bound by exactly this).
    if (x < a.tx && y < a.ty) return 0.0;
    return pow_kind(x, a.e_par, a.k_par) + pow_kind(y, a.e_perp, a.k_perp);
}

// arg-max over a warp with key (value descending, index ascending).  Values are margins: either -inf
// or >= 0, so their bit patterns order like unsigned integers (-inf and 0 both map to key 0: neither
// can win, only margins > 1 matter).  Three REDUX reductions (~100 cycles) instead of five rounds of
// three shuffles and a double compare (~350 cycles, measured).
__device__ __forceinline__ void warp_argmax_margin(double& v, int& i) {
    unsigned long long key = v > 0.0 ? (unsigned long long)__double_as_longlong(v) : 0ull;
    unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
    unsigned mhi = __reduce_max_sync(0xffffffffu, hi);
    unsigned mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? lo : 0u);
    unsigned mi = __reduce_min_sync(0xffffffffu, (hi == mhi && lo == mlo) ? (unsigned)i : 0xffffffffu);
    key = ((unsigned long long)mhi << 32) | mlo;
    v = key ? __longlong_as_double((long long)key) : -CUDART_INF;
    i = (int)mi;
}

#include "lattice.cuh"

// ------------------------------------------------------------------------------------------------
// A0: frame tables + hc validation
// ------------------------------------------------------------------------------------------------
__global__ void k_frame(int64_t N, int R, const double* __restrict__ angle, double* __restrict__ hc /* in: h_c, out: 1/h_c */,
                        double2* __restrict__ cs, int* __restrict__ flags) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    double sn, c;
    sincos(angle[i], &sn, &c);
    cs[i] = make_double2(c, sn);
    bool bad = !isfinite(angle[i]);
    for (int r = 0; r < R; ++r) {
        double h = hc[(int64_t)r * N + i];
        bad |= !(h > 0.0) || !isfinite(h);
        hc[(int64_t)r * N + i] = 1.0 / h;
    }
    if (bad) atomicOr(&flags[0], 1);
}

// ------------------------------------------------------------------------------------------------
// A1: cell grid
// ------------------------------------------------------------------------------------------------
__global__ void k_bbox(int64_t N, const double2* __restrict__ pos, double* __restrict__ bbox /*xmin,ymin,xmax,ymax*/) {
    __shared__ double sm[4][32];
    double xmin = CUDART_INF, ymin = CUDART_INF, xmax = -CUDART_INF, ymax = -CUDART_INF;
    bool bad = false;
    for (int64_t i = threadIdx.x; i < N; i += blockDim.x) {
        double2 p = pos[i];
        bad |= !isfinite(p.x) || !isfinite(p.y);
        xmin = fmin(xmin, p.x); xmax = fmax(xmax, p.x);
        ymin = fmin(ymin, p.y); ymax = fmax(ymax, p.y);
    }
    for (int o = 16; o > 0; o >>= 1) {
        xmin = fmin(xmin, __shfl_xor_sync(0xffffffffu, xmin, o));
        ymin = fmin(ymin, __shfl_xor_sync(0xffffffffu, ymin, o));
        xmax = fmax(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
        ymax = fmax(ymax, __shfl_xor_sync(0xffffffffu, ymax, o));
    }
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sm[0][w] = xmin; sm[1][w] = ymin; sm[2][w] = xmax; sm[3][w] = ymax; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int nw = blockDim.x >> 5;
        for (int k = 1; k < nw; ++k) {
            xmin = fmin(xmin, sm[0][k]); ymin = fmin(ymin, sm[1][k]);
            xmax = fmax(xmax, sm[2][k]); ymax = fmax(ymax, sm[3][k]);
        }
        bbox[0] = xmin; bbox[1] = ymin; bbox[2] = xmax; bbox[3] = ymax;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) bbox[0] = CUDART_NAN;
}

struct Grid { double x0, y0, inv_cell; int ncx, ncy; };

__device__ __forceinline__ void cell_xy(const Grid& g, double2 p, int& cx, int& cy) {
    cx = min(g.ncx - 1, max(0, (int)floor((p.x - g.x0) * g.inv_cell)));
    cy = min(g.ncy - 1, max(0, (int)floor((p.y - g.y0) * g.inv_cell)));
}

__global__ void k_cell_count(int64_t N, Grid g, const double2* __restrict__ pos, int* __restrict__ cell_of,
                             int* __restrict__ cell_cnt) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int cx, cy; cell_xy(g, pos[i], cx, cy);
    int c = cy * g.ncx + cx;
    cell_of[i] = c;
    atomicAdd(&cell_cnt[c], 1);
}

// single-CTA exclusive scan: cell_start[c] = sum_{c'<c} cnt[c'];  cell_start[ncells] = N
__global__ void k_cell_scan(int ncells, const int* __restrict__ cnt, int* __restrict__ start, int* __restrict__ fill) {
    __shared__ int wsum[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int base = 0; base < ncells; base += blockDim.x) {
        int c = base + threadIdx.x;
        int v = (c < ncells) ? cnt[c] : 0;
        int incl = v;
        for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
        if (lane == 31) wsum[w] = incl;
        __syncthreads();
        if (w == 0) {
            int t = (lane < nw) ? wsum[lane] : 0, inc2 = t;
            for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, inc2, o); if (lane >= o) inc2 += u; }
            wsum[lane] = inc2 - t;   // exclusive offsets of the warps
        }
        __syncthreads();
        int excl = carry + wsum[w] + incl - v;
        if (c < ncells) { start[c] = excl; fill[c] = excl; }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) start[ncells] = carry;
}

__global__ void k_cell_scatter(int64_t N, const int* __restrict__ cell_of, int* __restrict__ fill, int* __restrict__ items) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int slot = atomicAdd(&fill[cell_of[i]], 1);
    items[slot] = (int)i;      // order inside a cell is arbitrary; every ELL row is sorted afterwards
}

// degree of every spin; flags bit 1 = coincident pair.  One thread per spin over the 3x3 cells.
__global__ void k_count_neighbors(int64_t N, Grid g, double cut2, const double2* __restrict__ pos,
                                  const int* __restrict__ cell_start, const int* __restrict__ items,
                                  int* __restrict__ deg, int* __restrict__ flags, int* __restrict__ kmax,
                                  unsigned long long* __restrict__ total) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int d = 0;
    if (i < N) {
        double2 p = pos[i];
        int cx, cy; cell_xy(g, p, cx, cy);
        for (int yy = max(0, cy - 1); yy <= min(g.ncy - 1, cy + 1); ++yy)
            for (int xx = max(0, cx - 1); xx <= min(g.ncx - 1, cx + 1); ++xx) {
                int c = yy * g.ncx + xx;
                for (int q = cell_start[c]; q < cell_start[c + 1]; ++q) {
                    int j = items[q];
                    if (j == (int)i) continue;
                    double2 pj = pos[j];
                    double dx = p.x - pj.x, dy = p.y - pj.y;
                    double d2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
                    if (d2 == 0.0) atomicOr(&flags[0], 2);
                    else if (d2 <= cut2) ++d;
                }
            }
        deg[i] = d;
    }
    int m = d;
    unsigned long long sum = d;
    for (int o = 16; o > 0; o >>= 1) {
        m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicMax(kmax, m); atomicAdd(total, sum); }
}

// warp per spin: collect neighbours into shared memory, bitonic sort ascending, write the ELL row.
__global__ void k_fill_neighbors(int64_t N, Grid g, double cut2, int Kp, int Kp2,
                                 const double2* __restrict__ pos, const int* __restrict__ cell_start,
                                 const int* __restrict__ items, int* __restrict__ nbr) {
    extern __shared__ int sm_i[];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int* buf = sm_i + (size_t)w * Kp2;
    for (int64_t i = blockIdx.x * (int64_t)nw + w; i < N; i += (int64_t)gridDim.x * nw) {
        double2 p = pos[i];
        int cx, cy; cell_xy(g, p, cx, cy);
        int n = 0;
        for (int yy = max(0, cy - 1); yy <= min(g.ncy - 1, cy + 1); ++yy)
            for (int xx = max(0, cx - 1); xx <= min(g.ncx - 1, cx + 1); ++xx) {
                int c = yy * g.ncx + xx;
                int q0 = cell_start[c], q1 = cell_start[c + 1];
                for (int q = q0 + lane; q - lane < q1; q += 32) {
                    bool ok = false; int j = -1;
                    if (q < q1) {
                        j = items[q];
                        if (j != (int)i) {
                            double2 pj = pos[j];
                            double dx = p.x - pj.x, dy = p.y - pj.y;
                            double d2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
                            ok = (d2 != 0.0) && (d2 <= cut2);
                        }
                    }
                    unsigned m = __ballot_sync(0xffffffffu, ok);
                    if (ok) buf[n + __popc(m & ((1u << lane) - 1u))] = j;
                    n += __popc(m);
                }
            }
        for (int k = n + lane; k < Kp2; k += 32) buf[k] = 0x7fffffff;
        __syncwarp();
        for (int size = 2; size <= Kp2; size <<= 1)
            for (int stride = size >> 1; stride > 0; stride >>= 1) {
                for (int t = lane; t < (Kp2 >> 1); t += 32) {
                    int lo = 2 * t - (t & (stride - 1));       // index with bit `stride` cleared
                    int hi = lo + stride;
                    bool up = ((lo & size) == 0);
                    int a = buf[lo], b = buf[hi];
                    if ((a > b) == up) { buf[lo] = b; buf[hi] = a; }
                }
                __syncwarp();
            }
        int* row = nbr + i * (int64_t)Kp;
        for (int k = lane; k < Kp; k += 32) row[k] = (k < n) ? buf[k] : -1;
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------------
// A2: couplings.  Field at a from a unit moment at b, in a's fixed frame, times alpha (Eq. 3):
//     H = 3 r (m_b . r)/|r|^5 - m_b/|r|^3,  r = r_a - r_b;  (par, perp) = (H . m^_a, H . m^_a_perp)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 coupling(double2 pa, double2 ca, double2 pb, double2 cb, double alpha) {
    double dx = pa.x - pb.x, dy = pa.y - pb.y;
    double d2 = dx * dx + dy * dy;
    double inv = 1.0 / sqrt(d2);
    double inv3 = inv * inv * inv, inv5 = inv3 * inv * inv;
    double dot = cb.x * dx + cb.y * dy;
    double Hx = 3.0 * dx * dot * inv5 - cb.x * inv3;
    double Hy = 3.0 * dy * dot * inv5 - cb.y * inv3;
    return make_double2(alpha * (Hx * ca.x + Hy * ca.y), alpha * (-Hx * ca.y + Hy * ca.x));
}

__global__ void k_weights(int64_t N, int Kp, double alpha, const double2* __restrict__ pos,
                          const double2* __restrict__ cs, const int* __restrict__ nbr,
                          double2* __restrict__ w, double2* __restrict__ wT) {
    int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= N * Kp) return;
    int64_t i = t / Kp;
    int j = nbr[t];
    double2 a = make_double2(0.0, 0.0), b = a;
    if (j >= 0) {
        a = coupling(pos[i], cs[i], pos[j], cs[j], alpha);   // field at i from j
        b = coupling(pos[j], cs[j], pos[i], cs[i], alpha);   // field at j from i
    }
    w[t] = a;
    wT[t] = b;
}

// ------------------------------------------------------------------------------------------------
// A3: full gather.  G lanes cooperate on one ELL row; each lane takes 4 consecutive slots per step
// (one 16-byte index load + four 16-byte weight loads), partial sums folded with warp shuffles in a
// fixed order (deterministic).  blockIdx.y = replica.
// ------------------------------------------------------------------------------------------------
template <int G>
__global__ void __launch_bounds__(256) k_gather(int64_t N, int Kp, const int* __restrict__ nbr,
                                                const double2* __restrict__ w, const int8_t* __restrict__ s_all,
                                                double2* __restrict__ hdip_all) {
    asm volatile("griddepcontrol.launch_dependents;");   // lets a following k_scan become resident in this kernel's tail (see k_scan)
    const int8_t* __restrict__ s = s_all + (int64_t)blockIdx.y * N;
    double2* __restrict__ hdip = hdip_all + (int64_t)blockIdx.y * N;
    int64_t tid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int g = (int)(tid % G);
    const int64_t ngroups = (int64_t)gridDim.x * blockDim.x / G;
    const int64_t warp_first = (tid - (threadIdx.x & 31)) / G;      // group of lane 0: warp-uniform loop bound
    for (int64_t base = 0; warp_first + base < N; base += ngroups) {
        const int64_t i = tid / G + base;
        double ax = 0.0, ay = 0.0, bx = 0.0, by = 0.0;
        if (i < N) {
            const int4* rowi = reinterpret_cast<const int4*>(nbr + i * (int64_t)Kp);
            const double2* roww = w + i * (int64_t)Kp;
#pragma unroll 2
            for (int k4 = g; k4 < (Kp >> 2); k4 += G) {
                int4 j = __ldg(rowi + k4);
                const double2* ww = roww + 4 * k4;
                if (j.x >= 0) { double2 v = __ldg(ww + 0); double sj = (double)s[j.x]; ax = fma(sj, v.x, ax); ay = fma(sj, v.y, ay); }
                if (j.y >= 0) { double2 v = __ldg(ww + 1); double sj = (double)s[j.y]; bx = fma(sj, v.x, bx); by = fma(sj, v.y, by); }
                if (j.z >= 0) { double2 v = __ldg(ww + 2); double sj = (double)s[j.z]; ax = fma(sj, v.x, ax); ay = fma(sj, v.y, ay); }
                if (j.w >= 0) { double2 v = __ldg(ww + 3); double sj = (double)s[j.w]; bx = fma(sj, v.x, bx); by = fma(sj, v.y, by); }
            }
        }
        ax += bx; ay += by;
#pragma unroll
        for (int o = G >> 1; o > 0; o >>= 1) {
            ax += __shfl_xor_sync(0xffffffffu, ax, o);
            ay += __shfl_xor_sync(0xffffffffu, ay, o);
        }
        if (g == 0 && i < N) hdip[i] = make_double2(ax, ay);
    }
}

// ------------------------------------------------------------------------------------------------
// A4-A7: fused scan.  One thread per spin; writes hfix = rot(h_ext + h_th), the margin M and the
// arg-max of every leaf block of LB spins.  blockIdx.y = replica.
// ------------------------------------------------------------------------------------------------
struct FieldSpec { double sigma; uint64_t seed; uint32_t step; };

// rot(h_ext) + rot(h_th) of one spin in its own frame (Eq. 2 without h_dip; constant during a relaxation,
// PAPER.md:124).  One definition for k_scan and the in-CTA scan of the sweep kernel: identical rounding.
__device__ __forceinline__ double2 fixed_field(double2 c, double2 he, const FieldSpec& fs, int r, uint32_t i) {
    const double ex = he.x, ey = he.y;
    if (fs.sigma != 0.0) {
        double2 t = thermal_xy(fs.sigma, fs.seed + (uint64_t)r, fs.step, i);
        // (ext + th) rotated together would round differently from the paper's sum of three fields;
        // rotate separately and add (Eq. 2)
        double tp = t.x * c.x + t.y * c.y, tq = -t.x * c.y + t.y * c.x;
        double ep = ex * c.x + ey * c.y, eq = -ex * c.y + ey * c.x;
        return make_double2(ep + tp, eq + tq);
    }
    return make_double2(ex * c.x + ey * c.y, -ex * c.y + ey * c.x);
}

struct ScanGroup { double v; int idx; unsigned cnt; };  // result of one group of 32 scan CTAs
// uint32 words of scan scratch per replica: per-CTA counts, group tickets, group results
__host__ __device__ inline size_t scan_aux_stride(int ncta) { return 4 * (size_t)ncta + 4; }   // one ScanGroup per CTA

constexpr int SCAN_SPB_MIN = 512;                       // the smallest CTA span (sizes the per-CTA scratch)

// THREADS x SPT = SCAN_SPB consecutive spins per CTA (= SCAN_SPB / LB leaves): SPT spins per thread (independent load
// chains in flight).  1024 spins per CTA when a leaf is that large, else 512 (256-thread CTAs, four per SM: the CTA-wide
// barrier of the leaf reduction was the largest stall of the 512-thread version, profiles/r02_scan_cfg4.md).
template <int SCAN_SPT, int SCAN_SPB>
__global__ void __launch_bounds__(SCAN_SPB / SCAN_SPT) k_scan(int64_t N, int LB, Astroid ast, FieldSpec fs, int finalize,
                                               const double2* __restrict__ hext_all /*[R] (hx,hy)*/,
                                               const double2* __restrict__ cs, const double* __restrict__ hc_all,
                                               const int8_t* __restrict__ s_all, const double2* __restrict__ hdip_all,
                                               double2* __restrict__ hfix_all, double* __restrict__ M_all,
                                               double* __restrict__ bval_all, int* __restrict__ bidx_all, int nblk,
                                               unsigned* __restrict__ scnt_all /*[R][gridDim.x]*/, Counters* __restrict__ ctr,
                                               const double2* __restrict__ hloc /*[N] per-spin external field or NULL*/,
                                               int set_field, double2 field /*fs_set_field's pending global field, by value*/) {
    __shared__ double wv[32];                            // arg-max of every 32-spin slot of this CTA
    __shared__ int wi[32];
    __shared__ int is_last;
    const int r = blockIdx.y;
    const int64_t off = (int64_t)r * N;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    constexpr int SCAN_THREADS = SCAN_SPB / SCAN_SPT;
    const int64_t base = (int64_t)blockIdx.x * SCAN_SPB + threadIdx.x;
    // Programmatic dependent launch: this kernel may become resident while the gather kernel in front of it is still
    // running (the gathers call griddepcontrol.launch_dependents at their start, so that happens as soon as their last CTA
    // has started: in the tail of the gather, when SMs fall idle).  Until the wait below it reads only what no gather
    // writes (frames, 1/h_c): that cold-DRAM round trip and the launch latency overlap the gather's tail.  h_dip is
    // read, and everything is written, after the wait.  Behind any other kernel the wait falls through at once.
    asm volatile("griddepcontrol.launch_dependents;");   // a k_relax behind this scan may become resident (it waits at its top)
    double2 c[SCAN_SPT], hd[SCAN_SPT]; double ih[SCAN_SPT], sp[SCAN_SPT];
#pragma unroll
    for (int q = 0; q < SCAN_SPT; ++q) {
        const int64_t i = base + q * SCAN_THREADS;
        if (i < N) { c[q] = cs[i]; ih[q] = hc_all[off + i]; }
        else { c[q] = make_double2(1.0, 0.0); ih[q] = 1.0; }
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // fs_set_field launches nothing: its field arrives here by value, and one thread records it for the later readers
    const double2 he = set_field ? field : hext_all[r];
    if (set_field && blockIdx.x == 0 && threadIdx.x == 0) const_cast<double2*>(hext_all)[r] = field;
#pragma unroll
    for (int q = 0; q < SCAN_SPT; ++q) {
        const int64_t i = base + q * SCAN_THREADS;
        // the spins too: the kernel in front may be a relax kernel or fs_set_spins' fill, which write them
        if (i < N) { hd[q] = hdip_all[off + i]; sp[q] = (double)s_all[off + i]; } else { hd[q] = make_double2(0.0, 0.0); sp[q] = 1.0; }
    }
    unsigned long long nsw = 0;
#pragma unroll
    for (int q = 0; q < SCAN_SPT; ++q) {
        const int64_t i = base + q * SCAN_THREADS;
        double m = -CUDART_INF; int mi = 0x7fffffff;
        if (i < N) {
            double2 hei = he;                             // h_ext^(i) = global + per-spin
            if (hloc) { const double2 l = hloc[i]; hei = make_double2(he.x + l.x, he.y + l.y); }
            const double2 hf = fixed_field(c[q], hei, fs, r, (uint32_t)i);
            hfix_all[off + i] = hf;
            m = margin(hd[q].x + hf.x, hd[q].y + hf.y, sp[q], ih[q], ast);
            M_all[off + i] = m;
            mi = (int)i;
        }
        nsw += __popc(__ballot_sync(0xffffffffu, m > 1.0));
        warp_argmax_margin(m, mi);
        if (lane == 0) { wv[q * (SCAN_THREADS / 32) + w] = m; wi[q * (SCAN_THREADS / 32) + w] = mi; }   // slot = spin offset / 32
    }
    __syncthreads();
    {
        const int spl = LB >> 5, nleaf = SCAN_SPB / LB;  // 32-spin slots per leaf; leaves per CTA
        if ((int)threadIdx.x < nleaf) {
            const int s0 = threadIdx.x * spl;
            double bv = wv[s0]; int bi = wi[s0];
            for (int k = 1; k < spl; ++k) if (better(wv[s0 + k], wi[s0 + k], bv, bi)) { bv = wv[s0 + k]; bi = wi[s0 + k]; }
            const int blk = blockIdx.x * nleaf + threadIdx.x;
            if (blk < nblk) { bval_all[(int64_t)r * nblk + blk] = bv; bidx_all[(int64_t)r * nblk + blk] = bi; }
        }
    }
    if (!finalize) return;
    // A7 top level (fs_scan, and the hand-over count for k_relax_batch): every CTA publishes (its arg-max, its number
    // of switchable spins) and takes a ticket; the last CTA to finish reduces the <= N/1024 entries.  One dependent
    // round trip after the CTA's own work (a two-level version cost two).
    __shared__ unsigned wcnt[32];
    const int ncta = gridDim.x;
    ScanGroup* cres = reinterpret_cast<ScanGroup*>(scnt_all + (int64_t)r * scan_aux_stride(ncta));   // [ncta]
    if (lane == 0) wcnt[w] = (unsigned)nsw;
    __syncthreads();
    if (w == 0) {
        double v = lane < SCAN_SPB / 32 ? wv[lane] : -CUDART_INF;                  // SCAN_SPB / 32 slots of 32 spins
        int bi = lane < SCAN_SPB / 32 ? wi[lane] : 0x7fffffff;
        warp_argmax_margin(v, bi);
        unsigned c = lane < SCAN_THREADS / 32 ? wcnt[lane] : 0u;
        c = __reduce_add_sync(0xffffffffu, c);
        if (lane == 0) {
            cres[blockIdx.x].v = v; cres[blockIdx.x].idx = bi; cres[blockIdx.x].cnt = c;
            __threadfence();
            is_last = (atomicAdd(&ctr[r].ticket, 1u) == (unsigned)(ncta - 1));
        }
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double v = -CUDART_INF; int bi = 0x7fffffff;
    unsigned long long cnt = 0;
    for (int t = threadIdx.x; t < ncta; t += SCAN_THREADS) {
        const double tv = __ldcg(&cres[t].v); const int ti = __ldcg(&cres[t].idx);
        cnt += __ldcg(&cres[t].cnt);
        if (better(tv, ti, v, bi)) { v = tv; bi = ti; }
    }
    warp_argmax_margin(v, bi);
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    __shared__ unsigned long long wc[32];
    __syncthreads();                                     // wv/wi are reused
    if (lane == 0) { wv[w] = v; wi[w] = bi; wc[w] = cnt; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < SCAN_THREADS / 32; ++k) {
            if (better(wv[k], wi[k], v, bi)) { v = wv[k]; bi = wi[k]; }
            cnt += wc[k];
        }
        const bool any = v > 1.0;
        ctr[r].best_index = any ? bi : -1;
        ctr[r].best_L = any ? v : -CUDART_INF;
        ctr[r].n_switchable = (long long)cnt;
        ctr[r].ticket = 0u;
    }
}

// ------------------------------------------------------------------------------------------------
// A7-A9: relax loop.  One persistent CTA per replica; leaf-block maxima live in shared memory; per
// flip: top arg-max (shared memory) -> row k of the transposed ELL -> neighbours' h_dip -= 2 s_k w_ik
// (Eq. 3 is linear in s_k) -> margins of nbr(k) U {k} -> repair the touched leaf blocks.
// No host round trip and no grid-wide barrier per flip.
// ------------------------------------------------------------------------------------------------
#ifdef FS_RELAX_PROFILE
__device__ long long g_relax_prof[16];                  // cycles in: groups+top, update, barrier 1, leaf repair, barrier 2; flips
#define FS_PROF_T(var) long long var = clock64()
// behind a barrier: __syncthreads is BAR.SYNC.DEFER_BLOCKING, a clock read right after it sees the barrier's ISSUE; a
// volatile shared-memory read in between blocks until the barrier has completed, so the wait lands in the right phase
#define FS_PROF_TB(var) long long var; { const int prof_sink_ = *(volatile int*)&sh_stop; var = clock64() + (prof_sink_ & 0); }
#define FS_PROF_ADD(slot, a, b) prof[slot] += (b) - (a)
#else
#define FS_PROF_T(var)
#define FS_PROF_TB(var)
#define FS_PROF_ADD(slot, a, b)
#endif

// The arg-max hierarchy of the relax loop works on integer keys: key(M) = bit pattern of M if M > 0,
// else 0 (margins are -inf or >= 0, so keys order like the margins; only keys > key(1.0) can win).
typedef unsigned long long mkey_t;
__device__ __forceinline__ mkey_t margin_key(double m) { return m > 0.0 ? (mkey_t)__double_as_longlong(m) : 0ull; }
constexpr mkey_t KEY_ONE = 0x3ff0000000000000ull;      // key(1.0): "L > 1" (Eq. 5) <=> key > KEY_ONE

__device__ __forceinline__ void warp_argmax_key(mkey_t& key, int& i) {
    unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
    unsigned mhi = __reduce_max_sync(0xffffffffu, hi);
    unsigned mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? lo : 0u);
    unsigned mi = __reduce_min_sync(0xffffffffu, (hi == mhi && lo == mlo) ? (unsigned)i : 0xffffffffu);
    key = ((mkey_t)mhi << 32) | mlo;
    i = (int)mi;
}

// arg-max of 32 consecutive leaf maxima -> group maximum (one warp)
__device__ __forceinline__ void repair_group(int grp, int nblk, const mkey_t* bkey, const int* bidx, mkey_t* gkey, int* gidx_) {
    int t = grp * 32 + (threadIdx.x & 31);
    mkey_t v = t < nblk ? bkey[t] : 0ull;
    int i = t < nblk ? bidx[t] : 0x7fffffff;
    warp_argmax_key(v, i);
    if ((threadIdx.x & 31) == 0) { gkey[grp] = v; gidx_[grp] = i; }
}

#include "batch.cuh"

template <int RELAX_THREADS>                           // 512 (one big system per CTA) or 128 (ensembles of small systems)
__global__ void __launch_bounds__(RELAX_THREADS, RELAX_THREADS == 256 ? 4 : (RELAX_THREADS == 128 ? 8 : (RELAX_THREADS == 64 ? 16 : 1)))
k_relax(int64_t N, int Kp, int LBshift, int nblk, Astroid ast, long long max_flips, long long log_cap,
        const int* __restrict__ nbr, const double2* __restrict__ wT, const double* __restrict__ ihc_all,
        int8_t* __restrict__ s_all, double2* __restrict__ hdip_all, double2* __restrict__ hfix_all,
        double* __restrict__ M_all, const double* __restrict__ bval_all, const int* __restrict__ bidx_all,
        int* __restrict__ log_all, Counters* __restrict__ ctr,
        const int* __restrict__ cellidx /*NULL: no lattice*/, sgcell_t* __restrict__ sgrid, int64_t sgrid_stride,
        // sweep mode (T > 0): the CTA runs a whole field protocol, scanning its replica itself at every step
        int T, const double2* __restrict__ sweep_fields /*[T] (hx,hy)*/, FieldSpec fs, const double2* __restrict__ cs,
        long long* __restrict__ flips_per_step /*[R,T] or NULL*/, double2* __restrict__ hext_all,
        const double2* __restrict__ hloc /*[N] per-spin external field or NULL*/,
        const double* __restrict__ sweep_sigma /*[T] thermal std per step (annealing) or NULL*/,
        const double* __restrict__ sweep_lscale /*[T] scale of the static per-spin field per step or NULL*/,
        const double2* __restrict__ sweep_lseries /*[T,N] per-spin field per step or NULL*/,
        int use_base /*continue the flip count and log of k_relax_batch (ctr[r].batch_flips)*/,
        int state_smem /*the replica's per-spin state (h_dip, h_fix, M, 1/h_c, s: 49 B per spin) lives in shared memory*/) {
    // launched programmatically dependent on the k_scan in front of it (launch latency hidden): nothing is read before this
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // four-level arg-max hierarchy in shared memory:
    // spins -> leaves (LB spins) -> groups (32 leaves) -> supergroups (32 groups, <= 16 of them) -> top
    extern __shared__ unsigned char smem_raw[];
    const int ngrp = (nblk + 31) >> 5, nsup = (ngrp + 31) >> 5, LB = 1 << LBshift;
    mkey_t* bkey = reinterpret_cast<mkey_t*>(smem_raw);           // [nblk]
    mkey_t* gkey = bkey + nblk;                                   // [ngrp]
    mkey_t* skey = gkey + ngrp;                                   // [nsup]
    int* bidx = reinterpret_cast<int*>(skey + nsup);              // [nblk]
    int* gidx_ = bidx + nblk;                                     // [ngrp]
    int* sidx = gidx_ + ngrp;                                     // [nsup]
    int* touched = sidx + nsup;                                   // [Kp + 1] distinct leaf blocks touched by this flip
    __shared__ int sh_k, sh_sold, sh_stop, sh_ntouched;

    const int r = blockIdx.x;
    const int64_t off = (int64_t)r * N;
    const double* ihc = ihc_all + off;
    int8_t* s = s_all + off;
    double2* hdip = hdip_all + off;
    double2* hfix = hfix_all + off;
    double* M = M_all + off;
    int* flog = log_all + (int64_t)r * log_cap;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = RELAX_THREADS / 32;
    const bool one_warp = (Kp + 1 <= 32);               // the whole update fits one warp: no broadcast of k needed
    // Small replicas ("small N entirely in shared memory"): for the duration of a sweep the per-spin state is
    // staged into shared memory; every dependent round trip of the flip loop (neighbour state, margins, leaf rescan) then
    // costs a shared-memory access instead of an L2 one.  The couplings stay in global memory: read-only and the same for
    // all replicas of an SM, they hit in L1.  Written back at the end.
    double2 *g_hdip = hdip, *g_hfix = hfix; double* g_M = M; int8_t* g_s = s;
    if (state_smem) {
        unsigned char* sp = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(touched + Kp + 1) + 15) & ~(uintptr_t)15);
        double2* hd_s = reinterpret_cast<double2*>(sp); double2* hf_s = hd_s + N;
        double* M_s = reinterpret_cast<double*>(hf_s + N); double* ih_s = M_s + N; int8_t* s_s = reinterpret_cast<int8_t*>(ih_s + N);
        for (int64_t i = tid; i < N; i += RELAX_THREADS) { hd_s[i] = hdip[i]; hf_s[i] = hfix[i]; M_s[i] = M[i]; ih_s[i] = ihc[i]; s_s[i] = s[i]; }
        hdip = hd_s; hfix = hf_s; M = M_s; ihc = ih_s; s = s_s;
        __syncthreads();
    }

    long long nflips = use_base ? ctr[r].batch_flips : 0;
    const long long nflips0 = nflips;
    long long logpos = nflips % log_cap;
    int status = 0;
#ifdef FS_RELAX_PROFILE
    long long prof[12] = {0};
#endif
    int pf_row = -1, pf_done = -1;                      // prefetch engines: candidate whose row / state is in flight
    constexpr int PF_W0 = NW / 2;                       // warps PF_W0.. are prefetch engines at the top of every iteration
    const int nsteps = T > 0 ? T : 1;
    int st_last = 0;
    for (int st = 0; st < nsteps; ++st) {
    st_last = st;
    const long long nflips_before = nflips;
    if (T > 0) {
        // ---- A4-A7 inside the CTA (sweep mode): one warp per leaf, same arithmetic as k_scan
        const double2 he = sweep_fields[st];
        FieldSpec f2 = fs; f2.step = fs.step + (uint32_t)st;
        if (sweep_sigma) f2.sigma = sweep_sigma[st];
        for (int b = warp; b < nblk; b += NW) {
            mkey_t bv = 0ull; int bi = 0x7fffffff;
            for (int q = lane; q < LB; q += 32) {
                const int64_t i = ((int64_t)b << LBshift) + q;
                if (i < N) {
                    // h_ext^(i)(t) = global(t) + scale(t) * local_i + series(t, i)   (reading D-4)
                    double2 hei = he;
                    {
                        double lx = 0.0, ly = 0.0; bool anyl = false;
                        if (hloc) {
                            const double2 l = hloc[i];
                            if (sweep_lscale) { const double sc = sweep_lscale[st]; lx = __dmul_rn(sc, l.x); ly = __dmul_rn(sc, l.y); }
                            else { lx = l.x; ly = l.y; }
                            anyl = true;
                        }
                        if (sweep_lseries) {
                            const double2 l2 = sweep_lseries[(int64_t)st * N + i];
                            lx = anyl ? __dadd_rn(lx, l2.x) : l2.x; ly = anyl ? __dadd_rn(ly, l2.y) : l2.y;
                            anyl = true;
                        }
                        if (anyl) hei = make_double2(he.x + lx, he.y + ly);
                    }
                    const double2 hf = fixed_field(cs[i], hei, f2, r, (uint32_t)i);
                    hfix[i] = hf;
                    const double2 hd = hdip[i];
                    const double m = margin(hd.x + hf.x, hd.y + hf.y, (double)s[i], ihc[i], ast);
                    M[i] = m;
                    const mkey_t kv = margin_key(m);
                    if (kv > bv) { bv = kv; bi = (int)i; }
                }
            }
            warp_argmax_key(bv, bi);
            if (lane == 0) { bkey[b] = bv; bidx[b] = bi; }
        }
    } else {
        for (int t = tid; t < nblk; t += RELAX_THREADS) {
            bkey[t] = margin_key(bval_all[(int64_t)r * nblk + t]);
            bidx[t] = bidx_all[(int64_t)r * nblk + t];
        }
    }
    __syncthreads();
    for (int g = warp; g < ngrp; g += NW) repair_group(g, nblk, bkey, bidx, gkey, gidx_);
    __syncthreads();
    for (int g = warp; g < nsup; g += NW) repair_group(g, ngrp, gkey, gidx_, skey, sidx);
    if (tid == 0) { sh_stop = 0; sh_ntouched = 0; }
    __syncthreads();
    for (;;) {
        FS_PROF_T(c0);
        int k = 0, s_old = 0;
        if (warp == 0) {
            // ---- A7: top arg-max over the <= 8 supergroup maxima (warp 0)
            mkey_t v = lane < nsup ? skey[lane] : 0ull;
            k = lane < nsup ? sidx[lane] : 0x7fffffff;
            warp_argmax_key(v, k);
            bool stop = !(v > KEY_ONE);                 // no switchable spin left
            if (!stop && max_flips > 0 && nflips - nflips0 >= max_flips) { stop = true; status = 1; }
            if (stop) k = -1;
            if (lane == 0) { sh_k = k; sh_stop = stop ? 1 + status : 0; sh_ntouched = 0; }
        } else if (warp == 1 && one_warp && cellidx) {
            // Keep the stencil gather's spin grid in step.  The cell index of k is a dependent global load: issued after the
            // update barrier (as it was) it held the repair stage back by an L2 round trip; here an idle warp finds k itself
            // (the same arg-max as warp 0, no barrier between the two) and is done long before the update is.
            mkey_t v = lane < nsup ? skey[lane] : 0ull;
            int kk = lane < nsup ? sidx[lane] : 0x7fffffff;
            warp_argmax_key(v, kk);
            if (lane == 0 && v > KEY_ONE && !(max_flips > 0 && nflips - nflips0 >= max_flips))
                sgrid[(int64_t)r * sgrid_stride + cellidx[kk]] = (s[kk] > 0 ? SG_DOWN : SG_UP);   // s[k] is rewritten after the barrier
        } else if (warp >= PF_W0 && one_warp) {         // (with K + 1 > 32 every warp is needed for the update itself)
            // ---- prefetch engines (not on the critical path): the best spin of every 8th group is a likely
            // future flip.  Iteration n brings its ELL row to L2; iteration n+1 reads the row (an L2 hit by
            // then) and brings its neighbours' state, its coupling row and its own leaf of margins to L2.
            const int e = warp - PF_W0, ne = NW - PF_W0;
            if (pf_row >= 0 && !state_smem) {
                for (int t = lane; t < Kp; t += 32) {
                    int i = __ldcg(nbr + (int64_t)pf_row * Kp + t);
                    if (i >= 0) {
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(hdip + i));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(hfix + i));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(ihc + i));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(M + i));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(s + i));
                    }
                }
                for (int t = lane * 8; t < Kp; t += 256) asm volatile("prefetch.global.L2 [%0];" ::"l"(wT + (int64_t)pf_row * Kp + t));
                const int64_t lbase = ((int64_t)pf_row >> LBshift) << LBshift;
                for (int q = lane * 16; q < LB; q += 512)
                    if (lbase + q < N) asm volatile("prefetch.global.L2 [%0];" ::"l"(M + lbase + q));
                pf_done = pf_row; pf_row = -1;
            }
            mkey_t v = 0ull; int c = 0x7fffffff;
            for (int g = e + ne * lane; g < ngrp; g += ne * 32) {
                mkey_t kv = gkey[g]; int ki = gidx_[g];
                if (kv > v || (kv == v && ki < c)) { v = kv; c = ki; }
            }
            warp_argmax_key(v, c);
            if (v > KEY_ONE && c != pf_done) {
                for (int t = lane * 32; t < Kp; t += 1024) asm volatile("prefetch.global.L2 [%0];" ::"l"(nbr + (int64_t)c * Kp + t));
                pf_row = c;
            }
        }
        if (!one_warp) {
            __syncthreads();
            k = sh_k;
            if (tid == RELAX_THREADS - 32 && cellidx && k >= 0)  // (the last warp has the smallest share of the update)
                sgrid[(int64_t)r * sgrid_stride + cellidx[k]] = (s[k] > 0 ? SG_DOWN : SG_UP);
        }
        FS_PROF_T(c1);
        // ---- A8: flip k, update its neighbours incrementally, recompute their margins
        if (k >= 0 && (one_warp ? warp == 0 : true)) {
            const int* rowk = nbr + (int64_t)k * Kp;
            const double2* wTk = wT + (int64_t)k * Kp;
            s_old = s[k];                               // s[k] is rewritten only after the barrier below
            const double two_s = 2.0 * (double)s_old;
            for (int t0 = warp * 32; t0 <= Kp; t0 += RELAX_THREADS) {
                const int t = t0 + lane;
                int i = -1;
                if (t <= Kp) i = (t == Kp) ? k : rowk[t];        // entry Kp is the flipped spin itself
                int blk = -1;
                if (i >= 0) {
                    double2 hd = hdip[i], hf = hfix[i];
                    double si = (double)s[i], ih = ihc[i];
                    if (t == Kp) si = -(double)s_old;
                    else {
                        double2 wt = wTk[t];
                        hd.x -= two_s * wt.x;           // h_i -= 2 s_k,old alpha g_ik
                        hd.y -= two_s * wt.y;
                        hdip[i] = hd;
                    }
                    double m = margin(hd.x + hf.x, hd.y + hf.y, si, ih, ast);
                    M[i] = m;
                    blk = i >> LBshift;
                    // the leaf maximum can only change if i was its arg-max or reaches its value
                    const mkey_t nk = margin_key(m);
                    if (!(i == bidx[blk] || (nk != 0ull && nk >= bkey[blk]))) blk = -1;
                    if (m > 1.0 && t != Kp) {           // a likely next flip: bring its ELL rows to L2 now
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(nbr + (int64_t)i * Kp));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(wT + (int64_t)i * Kp));
                    }
                }
                // leaf blocks to rescan -> compact list.  Duplicates are harmless (the same leaf is rescanned
                // twice with the same result), so they are only removed cheaply: ELL rows are sorted, hence the
                // leaf index is non-decreasing along the lanes and a compare with the previous lane finds
                // nearly all repeats (a MATCH.ANY here cost ~450 cycles on the per-flip critical path).
                int prev = __shfl_up_sync(0xffffffffu, blk, 1);
                if (lane == 0) prev = -2;
                const bool leader = blk >= 0 && blk != prev;
                unsigned lead = __ballot_sync(0xffffffffu, leader);
                int base = 0;
                if (!one_warp) {
                    if (lane == 0 && lead) base = atomicAdd(&sh_ntouched, __popc(lead));
                    base = __shfl_sync(0xffffffffu, base, 0);
                }
                if (leader) touched[base + __popc(lead & ((1u << lane) - 1u))] = blk;
                if (one_warp && lane == 0) sh_ntouched = __popc(lead);
            }
            if (warp == 0 && lane == 0) sh_sold = s_old;
        }
        FS_PROF_T(c2);
        __syncthreads();
        FS_PROF_TB(c3);
        if (sh_stop) { status = sh_stop - 1; break; }
        if (tid == 0) {
            s[sh_k] = (int8_t)(-sh_sold);
            // ring buffer: the last log_cap flips are kept.  A running position: a 64-bit modulo here sits on the per-flip
            // critical path (this thread's warp rescans the first touched leaf next) and cost 0.4 us per flip
            flog[logpos] = sh_k; logpos = (logpos + 1 == log_cap) ? 0 : logpos + 1;
        }
        // ---- A7 repair, level by level, one warp per touched leaf (duplicated group work is harmless)
        const int ntouched = sh_ntouched;
        for (int t = warp; t < ntouched; t += NW) {
            const int blk = touched[t];
            mkey_t bv = 0ull; int bi = 0x7fffffff;
            const int64_t base = ((int64_t)blk << LBshift) + lane;
            for (int q0 = 0; q0 < LB; q0 += 256) {              // 8 independent loads in flight per lane
                double m[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    int64_t i = base + q0 + 32 * u;
                    m[u] = (q0 + 32 * u < LB && i < N) ? (state_smem ? M[i] : __ldcg(M + i)) : -CUDART_INF;
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    mkey_t kv = margin_key(m[u]);
                    if (kv > bv) { bv = kv; bi = (int)(base + q0 + 32 * u); }          // ascending index: strict > keeps the lowest
                }
            }
            warp_argmax_key(bv, bi);
            if (lane == 0) { bkey[blk] = bv; bidx[blk] = bi; }
        }
        FS_PROF_T(c3b);
        __syncthreads();
        FS_PROF_TB(c3c);
        for (int t = warp; t < ntouched; t += NW) repair_group(touched[t] >> 5, nblk, bkey, bidx, gkey, gidx_);
        __syncthreads();
        FS_PROF_TB(c3d);
        for (int t = warp; t < ntouched; t += NW) repair_group(touched[t] >> 10, ngrp, gkey, gidx_, skey, sidx);
        ++nflips;
        FS_PROF_T(c4);
        __syncthreads();
        FS_PROF_TB(c5);
        FS_PROF_ADD(0, c0, c1); FS_PROF_ADD(1, c1, c2); FS_PROF_ADD(2, c2, c3); FS_PROF_ADD(3, c3, c4); FS_PROF_ADD(4, c4, c5);
        FS_PROF_ADD(5, c3, c3b); FS_PROF_ADD(6, c3b, c3c); FS_PROF_ADD(7, c3c, c3d); FS_PROF_ADD(8, c3d, c4);
    }
    if (T > 0 && tid == 0 && flips_per_step) flips_per_step[(int64_t)r * T + st] = nflips - nflips_before;
    if (status) break;                                  // max_flips reached
    __syncthreads();                                    // the next step's scan rewrites the hierarchy
    }   // steps
    // a sweep stopped by max_flips leaves the fields of the step it actually reached (hfix, M and the spins
    // belong to that step) and zero flips for the steps it never ran
    if (state_smem) {
        __syncthreads();
        for (int64_t i = tid; i < N; i += RELAX_THREADS) { g_hdip[i] = hdip[i]; g_hfix[i] = hfix[i]; g_M[i] = M[i]; g_s[i] = s[i]; }
    }
    if (T > 0 && tid == 0) hext_all[r] = sweep_fields[st_last];
    if (T > 0 && flips_per_step)
        for (int t = st_last + 1 + tid; t < T; t += RELAX_THREADS) flips_per_step[(int64_t)r * T + t] = 0;
    if (tid == 0) {
        ctr[r].total_flips += nflips;
        ctr[r].last_flips = nflips;
        ctr[r].status = status;
        ctr[r].last_step = st_last;
#ifdef FS_RELAX_PROFILE
        for (int q = 0; q < 12; ++q) atomicAdd((unsigned long long*)&g_relax_prof[q], (unsigned long long)prof[q]);
        atomicAdd((unsigned long long*)&g_relax_prof[15], (unsigned long long)nflips);
#endif
    }
}

// ------------------------------------------------------------------------------------------------
// fs_get_fields
// ------------------------------------------------------------------------------------------------
__global__ void k_fields_out(int64_t N, int which, FieldSpec fs, const double2* __restrict__ hext_all,
                             const double2* __restrict__ cs, const double2* __restrict__ hdip_all,
                             double2* __restrict__ out_all, const double2* __restrict__ hloc) {
    int r = blockIdx.y;
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    double2 c = cs[i];
    double2 he = hext_all[r];
    if (hloc) { const double2 l = hloc[i]; he = make_double2(he.x + l.x, he.y + l.y); }
    double2 d = hdip_all[(int64_t)r * N + i];
    double2 e = make_double2(he.x * c.x + he.y * c.y, -he.x * c.y + he.y * c.x);
    double2 t = make_double2(0.0, 0.0);
    if (fs.sigma != 0.0 && (which == FS_FIELD_TOTAL || which == FS_FIELD_THERMAL)) {
        double2 g = thermal_xy(fs.sigma, fs.seed + (uint64_t)r, fs.step, (uint32_t)i);
        t = make_double2(g.x * c.x + g.y * c.y, -g.x * c.y + g.y * c.x);
    }
    double2 o;
    if (which == FS_FIELD_DIP) o = d;
    else if (which == FS_FIELD_EXT) o = e;
    else if (which == FS_FIELD_THERMAL) o = t;
    else o = make_double2(d.x + e.x + t.x, d.y + e.y + t.y);
    out_all[(int64_t)r * N + i] = o;
}

// ------------------------------------------------------------------------------------------------
// Analysis reductions of a (usually annealed) state.
// ------------------------------------------------------------------------------------------------
// Spin-spin correlation: "the correlation of two spins is defined as +1 (-1) if their dipole interaction is
// minimized (maximized)", as a function of their separation.  The pair energy is -s_i s_j g_par,ij (Eq. 3), so
// c_ij = sign(s_i s_j g_par,ij); pairs with |g_par| d^3 < 1e-9 (no parallel coupling) are skipped (reading D-5).
// Every unordered neighbour pair once; bin = floor(d / bin_width) from IEEE operations without contraction, so the
// integer bins equal the oracle's.  blockIdx.y = replica; counts by replica 0 only.
constexpr int CORR_MAX_BINS = 2048;
__global__ void __launch_bounds__(256) k_correlation(int64_t N, int Kp, double bin_width, int nbins, const double2* __restrict__ pos,
                                                     const double2* __restrict__ cs, const int* __restrict__ nbr,
                                                     const int8_t* __restrict__ s_all, long long* __restrict__ sum_all,
                                                     long long* __restrict__ count) {
    __shared__ int sh_sum[CORR_MAX_BINS];
    __shared__ int sh_cnt[CORR_MAX_BINS];
    const int r = blockIdx.y;
    const int8_t* s = s_all + (int64_t)r * N;
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) { sh_sum[b] = 0; sh_cnt[b] = 0; }
    __syncthreads();
    const int64_t total = N * (int64_t)Kp;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = t / Kp;
        const int j = nbr[t];
        if (j <= (int)i) continue;                       // padding (-1) and the mirrored entry
        const double2 pi = pos[i], pj = pos[j];
        const double dx = pi.x - pj.x, dy = pi.y - pj.y;
        const double d = __dsqrt_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)));
        const double fb = floor(__ddiv_rn(d, bin_width));
        if (!(fb < (double)nbins)) continue;
        const double2 g = coupling(pi, cs[i], pj, cs[j], 1.0);
        if (fabs(g.x) * (d * d * d) < 1e-9) continue;
        const int c = ((double)s[i] * (double)s[j] * g.x > 0.0) ? 1 : -1;
        atomicAdd(&sh_sum[(int)fb], c);
        if (r == 0) atomicAdd(&sh_cnt[(int)fb], 1);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) {
        if (sh_sum[b]) atomicAdd((unsigned long long*)&sum_all[(int64_t)r * nbins + b], (unsigned long long)(long long)sh_sum[b]);
        if (r == 0 && sh_cnt[b]) atomicAdd((unsigned long long*)&count[b], (unsigned long long)sh_cnt[b]);
    }
}

// Vertex populations: a vertex = four magnets around a point (square / pinwheel ASI).  A moment points into the
// vertex if m_i . (r_v - r_i) > 0, r_v = mean position.  0 or 4 in: Type IV; 1 or 3: Type III; 2: Type I if the
// two in-pointing magnets are opposite (net moment zero), Type II if adjacent (reading D-6).
__global__ void k_vertex_populations(int64_t N, int64_t V, const int* __restrict__ vert, const double2* __restrict__ pos,
                                     const double2* __restrict__ cs, const int8_t* __restrict__ s_all,
                                     long long* __restrict__ counts_all) {
    __shared__ int sh[4];
    const int r = blockIdx.y;
    const int8_t* s = s_all + (int64_t)r * N;
    if (threadIdx.x < 4) sh[threadIdx.x] = 0;
    __syncthreads();
    for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < V; v += (int64_t)gridDim.x * blockDim.x) {
        int q[4]; double2 p[4];
        double vx = 0.0, vy = 0.0;
#pragma unroll
        for (int a = 0; a < 4; ++a) { q[a] = vert[4 * v + a]; p[a] = pos[q[a]]; vx += p[a].x; vy += p[a].y; }
        vx *= 0.25; vy *= 0.25;
        int nin = 0; double inx = 0.0, iny = 0.0; bool first = true, opposite = false;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const double rx = vx - p[a].x, ry = vy - p[a].y;
            const double2 c = cs[q[a]];
            const double si = (double)s[q[a]];
            if (si * c.x * rx + si * c.y * ry > 0.0) {
                ++nin;
                if (first) { inx = rx; iny = ry; first = false; }
                else opposite = (inx * rx + iny * ry) < 0.0;
            }
        }
        const int type = (nin == 0 || nin == 4) ? 3 : ((nin == 1 || nin == 3) ? 2 : (opposite ? 0 : 1));
        atomicAdd(&sh[type], 1);
    }
    __syncthreads();
    if (threadIdx.x < 4 && sh[threadIdx.x])
        atomicAdd((unsigned long long*)&counts_all[(int64_t)r * 4 + threadIdx.x], (unsigned long long)sh[threadIdx.x]);
}

__global__ void k_set_field(int R, double hx, double hy, double2* hext) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < R) hext[r] = make_double2(hx, hy);
}

__global__ void k_fill_i8(int64_t n, int8_t v, int8_t* p) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

}  // namespace

// ================================================================================================
// host side
// ================================================================================================
struct fs_sim {
    int64_t N = 0; int R = 1; int K = 0, Kp = 4, LB = 32, nblk = 0, ncells = 0;
    int64_t n_inter = 0, log_cap = 0;
    fs_params p{};
    Astroid ast{};
    Grid grid{};
    cudaStream_t stream = nullptr;
    int device = 0;                 // the device current at fs_create; every entry point switches to it
    int sm_count = 148;
    // geometry
    double2 *pos = nullptr, *cs = nullptr, *w = nullptr, *wT = nullptr;
    int *nbr = nullptr, *deg = nullptr;
    // per replica
    double* hc = nullptr; int8_t* s = nullptr; double2 *hdip = nullptr, *hfix = nullptr; double* M = nullptr;
    double* bval = nullptr; int* bidx = nullptr; unsigned* scnt = nullptr; int* flog = nullptr; Counters* ctr = nullptr;
    double2* hext = nullptr;     // [R] device copy of the global field
    // state
    bool fields_dirty = true;
    double sigma = 0.0; uint64_t seed = 0; uint32_t step = 0;
    double2* hext_host = nullptr;   // pinned staging [R]
    bool field_pending = false;     // fs_set_field's value has not reached sim->hext yet: the next k_scan takes it by value
    double2 field_value{};
    Counters* ctr_host = nullptr;   // pinned staging [R]
    double2* hloc = nullptr;        // per-spin external field [N] in use (= hloc_buf), NULL = none
    double2* hloc_buf = nullptr;    // its place in the caller's workspace
    int gather_variant = FS_GATHER_AUTO;
    size_t relax_smem = 0;
    // regular-lattice stencil (lattice.cuh); library-owned device memory, freed by fs_destroy
    bool stencil_ok = false;
    int stencil_reason = 0;         // why not (FS_LATTICE_* code), 0 = active
    LatFrame lframe{};
    LatGrid lg{};
    void* lat_mem = nullptr;        // sub | cu | cv
    void* st_mem = nullptr;         // gidx | T | owner | rowtab | scratch
    uint8_t* lat_sub = nullptr; int *lat_cu = nullptr, *lat_cv = nullptr;
    sgcell_t* sgrid = nullptr; int* cellidx = nullptr; bool sgrid_valid = false;
    int* gidx = nullptr; double2* T = nullptr; unsigned long long* owner = nullptr; int2* rowtab = nullptr;
    float2* Tf = nullptr;           // fp32 copy of T (the optional fp32 field path)
    CUtensorMap sg_map{};           // TMA descriptor of the spin grids [R * nsub][Vpa][Upa], box = PU x SH x 1 (paired fp64 kernel)
    int st_nw = 4, st_rs = 1, st_pv = 0, st_ov = ST_OV; size_t st_smem = 0; bool st_ct = false;
    bool st_sym = false;            // inversion-paired stencil (c_prow / c_pstart tables below, host copies: they are tiny)
    std::vector<int4> prow; std::vector<int2> pstart; std::vector<int> ptofs, rtofs;
    unsigned long long st_id = 0;   // identity for the ownership of the constant-memory table
    double st_maxdev = 0.0, st_wmax = 0.0;
    long long st_slots = 0;         // stencil slots present (sum over sublattice pairs)
    // exact batched flips (batch.cuh); library-owned scratch, freed by fs_destroy
    void* bt_mem = nullptr; BatchArgs bt{}; bool bt_ok = false; int bt_P = 0, bt_alloc = 0, bt_seq = 64, bt_min_commit = 20, bt_max_chain = BT_LMAX, bt_grid = 0;
};

namespace {

struct GridPlan {
    Grid g; int ncells; double cut2;
};

struct Layout {
    // grid-phase buffers (depend on N, ncells only)
    size_t scratch, cell_of, cell_cnt, cell_start, cell_fill, items, deg;
    size_t grid_end;
    // K-dependent
    size_t pos, cs, nbr, w, wT, hc, s, hdip, hfix, M, bval, bidx, scnt, flog, ctr, hext, hloc, batch, total;
};

// Scratch of k_relax_batch (batch.cuh), carved from the caller's workspace.  The batched kernel applies to one large
// system with a moderate degree; elsewhere the region is empty.
struct BatchLayout { size_t ctl, owner, seeds, edges, ecount, npos, elems, undo, blocks, clist, cand, cbits, total; int Pdef, P; };
inline bool batch_applies(int64_t N, int R, int K) { return R == 1 && K >= 1 && K <= 64 && N >= 16384; }
int batch_default_seeds(int64_t N, int K) {
    const double p = 4.0 * std::sqrt((double)N / (double)(K + 1));
    return (int)std::max(64.0, std::min((double)BT_PMAX, std::floor(p)));
}
BatchLayout batch_layout(int64_t N, int K, int Kp) {
    // seeds per round: commits per round grow with the seeds, collisions between growing regions with their square;
    // measured optimum on config 4 at three sizes (125 k, 501 k, 2.0 M spins: 384-512, 768-1024, 1792-2048 seeds):
    // about 4 sqrt(N / (K + 1)).  Scratch is sized for twice that so that fs_set_batch can raise it.
    BatchLayout b{};
    b.Pdef = batch_default_seeds(N, K);
    b.P = std::min<int>(BT_PMAX, 2 * b.Pdef);
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    b.ctl = take(sizeof(BatchCtl)); b.owner = take(4 * (size_t)N); b.seeds = take(sizeof(BatchSeed) * BT_PMAX);
    b.edges = take(2 * (size_t)BT_PMAX * BT_EMAX); b.ecount = take(BT_PMAX); b.npos = take(4 * (size_t)BT_PMAX);
    b.elems = take(sizeof(BatchElem) * (size_t)b.P * BT_LMAX);
    b.undo = take(sizeof(BatchUndo) * (size_t)b.P * BT_LMAX * (size_t)(Kp + 1));
    b.blocks = take(sizeof(BatchBlock) * BT_PMAX); b.clist = take(sizeof(BatchCommit) * (size_t)b.P * BT_LMAX);
    b.cand = take(4 * (size_t)N); b.cbits = take(4 * (size_t)((N + 31) / 32));
    b.total = o;
    return b;
}

int choose_leaf(int64_t N, int* LB, int* nblk) {
    for (int lb = 32; lb <= 1024; lb <<= 1) {
        int64_t nb = (N + lb - 1) / lb;
        if (nb <= MAX_LEAF_BLOCKS) { *LB = lb; *nblk = (int)nb; return 0; }
    }
    return -1;
}

void layout_grid(Layout& L, int64_t N, int ncells) {
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    L.scratch = take(256);
    L.cell_of = take(sizeof(int) * N);
    L.cell_cnt = take(sizeof(int) * (size_t)(ncells + 1));
    L.cell_start = take(sizeof(int) * (size_t)(ncells + 1));
    L.cell_fill = take(sizeof(int) * (size_t)(ncells + 1));
    L.items = take(sizeof(int) * N);
    L.deg = take(sizeof(int) * N);
    L.grid_end = o;
}

void layout_rest(Layout& L, int64_t N, int R, int K, int Kp, int nblk, int64_t log_cap) {
    size_t o = L.grid_end;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    size_t NK = (size_t)N * Kp, RN = (size_t)R * N;
    L.pos = take(16 * (size_t)N);
    L.cs = take(16 * (size_t)N);
    L.nbr = take(4 * NK);
    L.w = take(16 * NK);
    L.wT = take(16 * NK);
    L.hc = take(8 * RN);
    L.s = take(RN);
    L.hdip = take(16 * RN);
    L.hfix = take(16 * RN);
    L.M = take(8 * RN);
    L.bval = take(8 * (size_t)R * nblk);
    L.bidx = take(4 * (size_t)R * nblk);
    L.flog = take(4 * (size_t)R * log_cap);
    L.scnt = take(4 * (size_t)R * scan_aux_stride((int)((N + SCAN_SPB_MIN - 1) / SCAN_SPB_MIN)));
    L.ctr = take(sizeof(Counters) * (size_t)R);
    L.hext = take(16 * (size_t)R);
    L.hloc = take(16 * (size_t)N);                       // per-spin external field of fs_set_local_field
    L.batch = take(batch_applies(N, R, K) ? batch_layout(N, K, Kp).total : 0);
    L.total = o;
}

int check_params(int64_t N, int R, const fs_params* p) {
    if (!p) return fail(FS_ERR_ARG, "params is NULL");
    if (N <= 0 || N > 0x7ffffff0LL) return fail(FS_ERR_ARG, "N=%lld out of range", (long long)N);
    if (R <= 0) return fail(FS_ERR_ARG, "R=%d must be positive", R);
    if (!(p->b > 0) || !(p->c > 0) || !(p->beta > 0) || !(p->gamma > 0) || !(p->neighbor_distance > 0) ||
        !std::isfinite(p->alpha) || !std::isfinite(p->neighbor_distance))
        return fail(FS_ERR_ARG, "b, c, beta, gamma, neighbor_distance must be > 0 and alpha finite");
    return FS_OK;
}

// bounding box -> cell grid plan.  `bbox_dev` = 4 doubles of device scratch.  Synchronises.
int plan_grid(int64_t N, const double* pos_dev, const fs_params* p, double* bbox_dev, cudaStream_t st, GridPlan* out) {
    k_bbox<<<1, 1024, 0, st>>>(N, reinterpret_cast<const double2*>(pos_dev), bbox_dev); LAUNCHED();
    double bb[4];
    CUDA_TRY(cudaMemcpyAsync(bb, bbox_dev, sizeof(bb), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (!(bb[0] == bb[0])) return fail(FS_ERR_ARG, "non-finite position");
    double cell = p->neighbor_distance * (1.0 + 1e-6);
    double ex = bb[2] - bb[0], ey = bb[3] - bb[1];
    // cap the number of cells at ~4N (sparse point sets / tiny cutoffs): larger cells stay correct
    for (;;) {
        double nx = std::floor(ex / cell) + 1.0, ny = std::floor(ey / cell) + 1.0;
        if (nx * ny <= 4.0 * (double)N + 1024.0) break;
        cell *= 1.5;
    }
    out->g.x0 = bb[0]; out->g.y0 = bb[1]; out->g.inv_cell = 1.0 / cell;
    out->g.ncx = (int)(std::floor(ex / cell) + 1.0);
    out->g.ncy = (int)(std::floor(ey / cell) + 1.0);
    out->ncells = out->g.ncx * out->g.ncy;
    out->cut2 = p->neighbor_distance * p->neighbor_distance * (1.0 + 1e-9);
    return FS_OK;
}

// cell grid + degree count inside `base` laid out by layout_grid.  Synchronises; returns K, I, flags.
int build_grid_and_count(int64_t N, const double* pos_dev, const GridPlan& gp, unsigned char* base, const Layout& L,
                         cudaStream_t st, int* K, long long* I, int* flags) {
    int* cell_of = (int*)(base + L.cell_of); int* cell_cnt = (int*)(base + L.cell_cnt);
    int* cell_start = (int*)(base + L.cell_start); int* cell_fill = (int*)(base + L.cell_fill);
    int* items = (int*)(base + L.items); int* deg = (int*)(base + L.deg);
    int* scr = (int*)(base + L.scratch);                 // [8]=flags, [9]=kmax, [10..11]=total (after 4 bbox doubles)
    const double2* pos = reinterpret_cast<const double2*>(pos_dev);
    CUDA_TRY(cudaMemsetAsync(cell_cnt, 0, sizeof(int) * (size_t)(gp.ncells + 1), st));
    CUDA_TRY(cudaMemsetAsync(scr + 9, 0, 3 * sizeof(int), st));    // kmax + total (flags keep k_frame's bits)
    int nb = (int)((N + 255) / 256);
    k_cell_count<<<nb, 256, 0, st>>>(N, gp.g, pos, cell_of, cell_cnt); LAUNCHED();
    k_cell_scan<<<1, 1024, 0, st>>>(gp.ncells, cell_cnt, cell_start, cell_fill); LAUNCHED();
    k_cell_scatter<<<nb, 256, 0, st>>>(N, cell_of, cell_fill, items); LAUNCHED();
    k_count_neighbors<<<nb, 256, 0, st>>>(N, gp.g, gp.cut2, pos, cell_start, items, deg, scr + 8, scr + 9,
                                          (unsigned long long*)(scr + 10)); LAUNCHED();
    int host[4];
    CUDA_TRY(cudaMemcpyAsync(host, scr + 8, sizeof(host), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    *flags = host[0]; *K = host[1];
    unsigned long long tot; std::memcpy(&tot, host + 2, 8); *I = (long long)tot;
    return FS_OK;
}

int pad_k(int K) { int kp = (K + 3) / 4 * 4; return kp < 4 ? 4 : kp; }

template <int G>
void launch_gather_g(fs_sim* sim) {
    int occ = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_gather<G>, 256, 0);
    if (occ < 1) occ = 1;
    int64_t groups_per_block = 256 / G;
    int64_t need = (sim->N + groups_per_block - 1) / groups_per_block;
    int64_t blocks = std::min<int64_t>(need, (int64_t)sim->sm_count * occ * 4);
    dim3 grid((unsigned)blocks, (unsigned)sim->R);
    k_gather<G><<<grid, 256, 0, sim->stream>>>(sim->N, sim->Kp, sim->nbr, sim->w, sim->s, sim->hdip);
    LAUNCHED();
}

int do_gather_stencil(fs_sim* sim) {
    const LatGrid& g = sim->lg;
    int TV = sim->st_ov * sim->st_nw;
    dim3 sgrid((unsigned)((g.Up + 31) / 32), (unsigned)((g.Vp + 31) / 32), (unsigned)g.nsub);
    if (!sim->sgrid_valid) {                             // the relax loop keeps the grids in step with its flips
        k_spin_grid<<<sgrid, 256, 0, sim->stream>>>(sim->N, g, sim->R, sim->gidx, sim->s, sim->sgrid);
        LAUNCHED();
        sim->sgrid_valid = true;
    }
    dim3 grid((unsigned)((g.U + ST_TU - 1) / ST_TU), (unsigned)((g.V + TV - 1) / TV), (unsigned)(g.nsub * sim->R));
    int threads = 32 * sim->st_nw * sim->st_rs;
#define FS_STENCIL_ARGS sim->N, g, sim->st_nw, sim->st_pv, sim->gidx, sim->sgrid, sim->T, sim->rowtab, sim->hdip
#define FS_LAUNCH_STENCIL1(MAXT, MINB, CTV, OVV)                                                                     \
    do {                                                                                                             \
        if (sim->st_pv == 64) k_gather_stencil<MAXT, MINB, CTV, OVV, false, 64><<<grid, threads, sim->st_smem, sim->stream>>>(FS_STENCIL_ARGS); \
        else k_gather_stencil<MAXT, MINB, CTV, OVV, false, 128><<<grid, threads, sim->st_smem, sim->stream>>>(FS_STENCIL_ARGS);                  \
    } while (0)
#define FS_LAUNCH_STENCIL_SYM(MAXT, MINB)                                                                            \
    do {                                                                                                             \
        if (sim->st_pv == 64) k_gather_stencil<MAXT, MINB, true, 8, true, 64><<<grid, threads, sim->st_smem, sim->stream>>>(FS_STENCIL_ARGS); \
        else k_gather_stencil<MAXT, MINB, true, 8, true, 128><<<grid, threads, sim->st_smem, sim->stream>>>(FS_STENCIL_ARGS);                  \
    } while (0)
    // 8 outputs per thread: 72 (<= 128 threads) or 80 registers.  A 16-output variant (128 registers, half the
    // window set-ups per DFMA) was measured at 64.4 us against 63.3 us on config 5 and is not instantiated.
#define FS_LAUNCH_STENCIL(CTV)                                                                      \
    do {                                                                                            \
        if (threads <= 128) FS_LAUNCH_STENCIL1(128, 7, CTV, 8);                                     \
        else FS_LAUNCH_STENCIL1(256, 3, CTV, 8);                                                    \
    } while (0)
    const bool f32 = sim->gather_variant == FS_GATHER_STENCIL_F32;
    if (sim->st_ct) {
        // the constant-memory table is shared by all simulations of the process (and by the fp64 / fp32 formats of one
        // simulation): take it over if needed
        std::lock_guard<std::mutex> lock(g_ct_mutex);
        unsigned long long& g_ct_owner = g_ct_owner_dev[sim->device & 63];
        cudaEvent_t& g_ct_event = g_ct_event_dev[sim->device & 63];
        const unsigned long long want = 2 * sim->st_id + (f32 ? 1 : 0);
        if (g_ct_owner != want) {
            if (g_ct_event) CUDA_TRY(cudaStreamWaitEvent(sim->stream, g_ct_event, 0));   // previous owner's kernels first
            const size_t nT = (size_t)g.nsub * g.nsub * g.W * g.H;
            if (f32) CUDA_TRY(cudaMemcpyToSymbolAsync(c_T, sim->Tf, 8 * nT, 0, cudaMemcpyDeviceToDevice, sim->stream));
            else CUDA_TRY(cudaMemcpyToSymbolAsync(c_T, sim->T, 16 * nT, 0, cudaMemcpyDeviceToDevice, sim->stream));
            CUDA_TRY(cudaMemcpyToSymbolAsync(c_rows, sim->rowtab, 8 * (size_t)g.nsub * g.nsub * g.W, 0,
                                             cudaMemcpyDeviceToDevice, sim->stream));
            CUDA_TRY(cudaMemcpyToSymbolAsync(c_rtofs, sim->rtofs.data(), 4 * sim->rtofs.size(), 0, cudaMemcpyHostToDevice, sim->stream));
            if (sim->st_sym) {
                CUDA_TRY(cudaMemcpyToSymbolAsync(c_sg_map, &sim->sg_map, sizeof(CUtensorMap), 0, cudaMemcpyHostToDevice, sim->stream));
                CUDA_TRY(cudaMemcpyToSymbolAsync(c_ptofs, sim->ptofs.data(), 4 * sim->ptofs.size(), 0, cudaMemcpyHostToDevice, sim->stream));
                CUDA_TRY(cudaMemcpyToSymbolAsync(c_prow, sim->prow.data(), 16 * sim->prow.size(), 0, cudaMemcpyHostToDevice, sim->stream));
                CUDA_TRY(cudaMemcpyToSymbolAsync(c_pstart, sim->pstart.data(), 8 * sim->pstart.size(), 0, cudaMemcpyHostToDevice, sim->stream));
            }
            g_ct_owner = want;
        }
        const bool sym = sim->st_sym && sim->gather_variant != FS_GATHER_STENCIL_PLAIN;
        if (f32) {
#define FS_LAUNCH_F32(MAXT, MINB, SYMV)                                                                              \
    do {                                                                                                             \
        if (sim->st_pv == 64) k_gather_stencil<MAXT, MINB, true, 8, SYMV, 64, float><<<grid, threads, sim->st_smem, sim->stream>>>(FS_STENCIL_ARGS); \
        else k_gather_stencil<MAXT, MINB, true, 8, SYMV, 128, float><<<grid, threads, sim->st_smem, sim->stream>>>(FS_STENCIL_ARGS);                  \
    } while (0)
            if (sym) { if (threads <= 128) FS_LAUNCH_F32(128, 7, true); else FS_LAUNCH_F32(256, 3, true); }
            else { if (threads <= 128) FS_LAUNCH_F32(128, 7, false); else FS_LAUNCH_F32(256, 3, false); }
#undef FS_LAUNCH_F32
        } else if (sym) {
            if (threads <= 128) FS_LAUNCH_STENCIL_SYM(128, 4); else FS_LAUNCH_STENCIL_SYM(256, 2);
        } else
        FS_LAUNCH_STENCIL(true);
        if (!g_ct_event) CUDA_TRY(cudaEventCreateWithFlags(&g_ct_event, cudaEventDisableTiming));
        CUDA_TRY(cudaEventRecord(g_ct_event, sim->stream));
    } else {
        FS_LAUNCH_STENCIL(false);
    }
#undef FS_LAUNCH_STENCIL
#undef FS_LAUNCH_STENCIL_SYM
#undef FS_STENCIL_ARGS
#undef FS_LAUNCH_STENCIL1
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    sim->fields_dirty = false;
    return FS_OK;
}

// Shape of the stencil kernel for this lattice: NW v-slabs x RS row groups per CTA.  Small model: every
// CTA does work ~ NW; an SM runs ceil(ctas / SMs) of them (one wave if they fit) and needs >= 20
// resident warps to keep its FP64 pipe busy.  Ties go to the larger tile (less halo), then fewer groups.
struct StencilShape { int nw, rs, pv, ov; size_t smem; };

bool stencil_ct(const LatGrid& g) {
    return (int64_t)g.nsub * g.nsub * g.W * g.H <= CT_MAX && g.nsub * g.nsub * g.W <= CR_MAX;
}

int stencil_pu(const LatGrid& g) { return ((ST_TU + 2 * g.Ru + 3) & ~3) <= 64 ? 64 : 128; }   // shared-memory row pitch (cells)

size_t stencil_smem(const LatGrid& g, int nw, int rs, int ov, int* pv_out) {
    int TV = ov * nw, SH = TV + 2 * g.Rv, pu = stencil_pu(g);
    size_t tsm = stencil_ct(g) ? 0 : 16 * (size_t)g.nsub * g.W * g.H;
    size_t tables = (tsm + 8 * (size_t)g.nsub * g.W + 128 * (size_t)TV + 8 + 127) & ~(size_t)127;   // the tiles are 128-byte aligned (TMA); 8 bytes in front of them hold its mbarrier
    // one spare row in front and behind: the sliding windows read one cell past the last slot of a row
    size_t tiles = 4 * (size_t)(g.nsub * SH + 1) * pu, red = (size_t)(rs - 1) * nw * 512 * ov;
    if (pv_out) *pv_out = pu;
    return tables + std::max(tiles, red);
}

bool plan_stencil(const fs_sim* sim, const LatGrid& g, StencilShape* out) {
    double best = 1e300; bool found = false;
    const int ov = ST_OV;
    for (int nw = 8; nw >= 1; nw >>= 1)
        for (int rs = 1; rs <= 4 && nw * rs <= (ov == 16 ? 4 : 8); rs <<= 1) {
            if (rs > g.W) continue;
            int pv; size_t smem = stencil_smem(g, nw, rs, ov, &pv);
            if (smem > 200 * 1024) continue;
            int threads = 32 * nw * rs, TV = ov * nw;
            int64_t ctas = (int64_t)((g.U + ST_TU - 1) / ST_TU) * ((g.V + TV - 1) / TV) * g.nsub * sim->R;
            int regs = ov == 16 ? 128 : (threads <= 128 ? 72 : 80);
            int64_t resident = std::min<int64_t>(std::min<int64_t>(65536 / (regs * threads), (227 * 1024) / (int64_t)(smem + 1024)),
                                                 std::min<int64_t>(2048 / threads, 32));
            if (resident < 1) continue;
            int64_t per_sm = (ctas + sim->sm_count - 1) / sim->sm_count;
            int64_t waves = (per_sm + resident - 1) / resident;
            double warps = (double)std::min(per_sm, resident) * nw * rs;
            double eff = std::min(1.0, warps * (ov / 8) / 20.0);     // a 16-output warp carries twice the independent DFMAs
            // multi-wave launches pay for a partly filled last wave
            double cost = (waves == 1 ? (double)per_sm : (double)waves * resident) * nw * (ov / 8) / eff;
            // reduction epilogue; halo staging per output; per-row window set-up per output
            cost *= 1.0 + 0.02 * (rs - 1) + 0.16 * 8 / (nw * ov) + (ov == 16 ? 0.0 : 0.10);
            if (cost < best - 1e-9) { best = cost; *out = StencilShape{nw, rs, pv, ov, smem}; found = true; }
        }
    return found;
}

int do_gather(fs_sim* sim) {
    bool stencil = sim->stencil_ok && sim->gather_variant != FS_GATHER_ELL_F64;
    if (stencil) return do_gather_stencil(sim);
    int q = sim->Kp / 4;
    if (q <= 1) launch_gather_g<1>(sim);
    else if (q <= 2) launch_gather_g<2>(sim);
    else if (q <= 4) launch_gather_g<4>(sim);
    else if (q <= 8) launch_gather_g<8>(sim);
    else if (q <= 16) launch_gather_g<16>(sim);
    else launch_gather_g<32>(sim);
    CUDA_TRY(cudaGetLastError());
    sim->fields_dirty = false;
    return FS_OK;
}

// ---- lattice detection (host logic + lattice.cuh kernels).  Never fails the creation: any problem
// leaves sim->stencil_ok = false with a reason code and the ELL gather in charge.
struct PickRow { double px, py, cx, cy; };

__global__ void k_lat_pick(int i0, int Kp, const int* __restrict__ nbr, const double2* __restrict__ pos,
                           const double2* __restrict__ cs, PickRow* __restrict__ out) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > Kp) return;
    int j = (t == Kp) ? i0 : nbr[(int64_t)i0 * Kp + t];
    PickRow r{0, 0, 2, 2};                               // (2,2) marks padding
    if (j >= 0) { double2 p = pos[j], c = cs[j]; r = PickRow{p.x, p.y, c.x, c.y}; }
    out[t] = r;
}

int lattice_fail(fs_sim* sim, int reason) {
    sim->stencil_ok = false; sim->stencil_reason = reason;
    if (sim->st_mem) { cudaFree(sim->st_mem); sim->st_mem = nullptr; }
    if (sim->lat_mem) { cudaFree(sim->lat_mem); sim->lat_mem = nullptr; }
    cudaGetLastError();
    return FS_OK;
}

// Inversion pairing of the stencil slots (lattice.cuh, SYM variant).  Eq. 3 is even in r_ij, so on a lattice
// with an inversion centre on the sites of sublattice si the slot (du, dv) of the pair (si, sj) has a partner
// (-du - cu, -dv - cv) with the same coupling.  (cu, cv) is searched in [-2, 2]^2 and accepted only if every
// present slot has a present partner whose table entry is BIT-IDENTICAL; otherwise the plain variant stays.
int build_inversion_pairs(fs_sim* sim, const LatGrid& g, const std::vector<unsigned long long>& own) {
    const int nsub = g.nsub, W = g.W, H = g.H, wh = W * H;
    std::vector<double2> T((size_t)nsub * nsub * wh);
    CUDA_TRY(cudaMemcpyAsync(T.data(), sim->T, 16 * T.size(), cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    std::vector<int4> prow; std::vector<int> ptofs; std::vector<int2> pstart((size_t)NSUB_MAX * NSUB_MAX, make_int2(0, 0));
    auto present = [&](int pair, int du, int dv) {
        if (du < -g.Ru || du > g.Ru || dv < -g.Rv || dv > g.Rv) return false;
        return own[(size_t)pair * wh + (size_t)(du + g.Ru) * H + (dv + g.Rv)] != ~0ull;
    };
    auto entry = [&](int pair, int du, int dv) { return T[(size_t)pair * wh + (size_t)(du + g.Ru) * H + (dv + g.Rv)]; };
    for (int pair = 0; pair < nsub * nsub; ++pair) {
        int fcu = 0, fcv = 0; bool found = false, any = false;
        for (int du = -g.Ru; du <= g.Ru && !any; ++du) for (int dv = -g.Rv; dv <= g.Rv; ++dv) if (present(pair, du, dv)) { any = true; break; }
        if (!any) { pstart[pair] = make_int2((int)prow.size(), 0); continue; }
        for (int cu = -2; cu <= 2 && !found; ++cu)
            for (int cv = -2; cv <= 2 && !found; ++cv) {
                bool ok = true;
                for (int du = -g.Ru; du <= g.Ru && ok; ++du)
                    for (int dv = -g.Rv; dv <= g.Rv && ok; ++dv) {
                        if (!present(pair, du, dv)) continue;
                        const int pu = -du - cu, pv = -dv - cv;
                        if (!present(pair, pu, pv) || (pu == du && pv == dv)) { ok = false; break; }
                        const double2 a = entry(pair, du, dv), b = entry(pair, pu, pv);
                        ok = a.x == b.x && a.y == b.y;               // equal values (+0 == -0: the products are the same)
                    }
                if (ok) { fcu = cu; fcv = cv; found = true; }
            }
        if (!found) return FS_OK;                        // no exact pairing: plain variant
        const int first = (int)prow.size();
        for (int du = g.Ru; du >= -g.Ru; --du) {
            const int pu = -du - fcu;
            if (pu > du) continue;                       // visited from the partner row
            // slots of row du to visit: all present ones, or (row paired with itself) those with dv > -dv - cv
            int a = 0, b = -1; bool anyrow = false;
            for (int dv = -g.Rv; dv <= g.Rv; ++dv)
                if (present(pair, du, dv) && (pu != du || 2 * dv > -fcv)) { if (!anyrow) a = dv; b = dv; anyrow = true; }
            if (!anyrow) continue;
            // holes inside [a, b] carry zero weight and must be holes in the mirrored row as well
            for (int dv = a; dv <= b; ++dv)
                if (present(pair, du, dv) != present(pair, pu, -dv - fcv)) return FS_OK;
            if (-b - fcv < -g.Rv || -a - fcv > g.Rv) return FS_OK;
            prow.push_back(make_int4((du + g.Ru) | ((pu + g.Ru) << 16), a, b, -a - fcv));
            ptofs.push_back(pair * wh + (du + g.Ru) * H + (a + g.Rv));
        }
        pstart[pair] = make_int2(first, (int)prow.size() - first);
    }
    if (prow.size() > (size_t)CP_MAX) return FS_OK;
    sim->prow = prow; sim->pstart = pstart; sim->ptofs = ptofs; sim->st_sym = true;
    return FS_OK;
}

// TMA descriptor of the spin grids for k_gather_stencil's paired fp64 variant: uint32 [R * nsub][Vpa][Upa] (u fastest),
// box = (shared-memory row pitch) x (tile rows + halo) x 1, no swizzle, zero fill outside.  cuTensorMapEncodeTiled is a
// driver call: its entry point is fetched through the runtime, so the library does not link against libcuda.
bool make_spin_grid_map(fs_sim* sim, const LatGrid& g) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) { cudaGetLastError(); return false; }
    const int SH = sim->st_ov * sim->st_nw + 2 * g.Rv, pu = sim->st_pv;
    if (SH > 256 || pu > 256) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.Upa, (cuuint64_t)g.Vpa, (cuuint64_t)sim->R * g.nsub};
    const cuuint64_t strides[2] = {(cuuint64_t)g.Upa * sizeof(sgcell_t), (cuuint64_t)g.Upa * g.Vpa * sizeof(sgcell_t)};
    const cuuint32_t box[3] = {(cuuint32_t)pu, (cuuint32_t)SH, 1u};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = ((encode_fn)fn)(&sim->sg_map, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, sim->sgrid, dims, strides, box, estr,
                                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

int detect_lattice(fs_sim* sim) {
    const int64_t N = sim->N; const int Kp = sim->Kp; cudaStream_t st = sim->stream;
    if (sim->K <= 0) return lattice_fail(sim, FS_LATTICE_NO_NEIGHBORS);
    // reference spin: lowest index among the spins of maximum degree (an interior spin)
    std::vector<int> deg((size_t)N);
    CUDA_TRY(cudaMemcpyAsync(deg.data(), sim->deg, 4 * (size_t)N, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    int i0 = 0;
    for (int64_t i = 1; i < N; ++i) if (deg[i] > deg[i0]) i0 = (int)i;
    // its neighbours' positions and orientations
    PickRow* pick_dev = nullptr;
    CUDA_TRY(cudaMalloc(&pick_dev, sizeof(PickRow) * (size_t)(Kp + 1)));
    k_lat_pick<<<(Kp + 1 + 127) / 128, 128, 0, st>>>(i0, Kp, sim->nbr, sim->pos, sim->cs, pick_dev); LAUNCHED();
    std::vector<PickRow> pick((size_t)Kp + 1);
    cudaError_t e = cudaMemcpyAsync(pick.data(), pick_dev, sizeof(PickRow) * (size_t)(Kp + 1), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(pick_dev);
    if (e != cudaSuccess) return fail(FS_ERR_CUDA, "lattice pick: %s", cudaGetErrorString(e));
    const PickRow me = pick[Kp];
    struct Nb { double dx, dy, cx, cy, len; };
    std::vector<Nb> nb;
    for (int t = 0; t < Kp; ++t)
        if (pick[t].cx <= 1.5) {
            double dx = pick[t].px - me.px, dy = pick[t].py - me.py;
            nb.push_back(Nb{dx, dy, pick[t].cx, pick[t].cy, std::sqrt(dx * dx + dy * dy)});
        }
    std::sort(nb.begin(), nb.end(), [](const Nb& a, const Nb& b) { return a.len < b.len; });
    // candidate lattice vectors: displacements to same-orientation neighbours, and differences of
    // displacements between neighbours that share an orientation (nearest 64 only)
    auto same = [](double ax, double ay, double bx, double by) { return std::fabs(ax - bx) < 1e-9 && std::fabs(ay - by) < 1e-9; };
    struct Vec { double x, y, len, ang; };
    std::vector<Vec> cand;
    auto push = [&](double x, double y) {
        double len = std::sqrt(x * x + y * y);
        if (!(len > 1e-9)) return;
        if (x < -1e-12 * len || (std::fabs(x) <= 1e-12 * len && y < 0)) { x = -x; y = -y; }   // half plane
        cand.push_back(Vec{x, y, len, std::atan2(y, x)});
    };
    for (const Nb& a : nb) if (same(a.cx, a.cy, me.cx, me.cy)) push(a.dx, a.dy);
    size_t near = std::min<size_t>(nb.size(), 64);
    for (size_t a = 0; a < near; ++a)
        for (size_t b = a + 1; b < near; ++b)
            if (same(nb[a].cx, nb[a].cy, nb[b].cx, nb[b].cy)) push(nb[a].dx - nb[b].dx, nb[a].dy - nb[b].dy);
    if (cand.empty()) return lattice_fail(sim, FS_LATTICE_NO_BASIS);
    std::sort(cand.begin(), cand.end(), [](const Vec& a, const Vec& b) {
        if (std::fabs(a.len - b.len) > 1e-9 * std::max(a.len, b.len)) return a.len < b.len;
        return std::fabs(a.ang) < std::fabs(b.ang);     // among equals: closest to the +x axis (spin index order)
    });
    const Vec a1 = cand[0];
    Vec a2{-a1.y, a1.x, a1.len, 0.0};                    // 1-D chains: any perpendicular
    for (const Vec& c : cand) {
        double cr = a1.x * c.y - a1.y * c.x;
        if (std::fabs(cr) > 1e-6 * a1.len * c.len) { a2 = c; if (cr < 0) { a2.x = -c.x; a2.y = -c.y; } break; }
    }
    double det = a1.x * a2.y - a1.y * a2.x;
    if (!(std::fabs(det) > 1e-12)) return lattice_fail(sim, FS_LATTICE_NO_BASIS);
    sim->lframe = LatFrame{me.px, me.py, a2.y / det, -a2.x / det, -a1.y / det, a1.x / det};

    // sublattices: one pass per sublattice
    CUDA_TRY(cudaMalloc(&sim->lat_mem, align_up((size_t)N) + 2 * align_up(4 * (size_t)N) + 256));
    unsigned char* lb = (unsigned char*)sim->lat_mem;
    sim->lat_sub = lb; sim->lat_cu = (int*)(lb + align_up((size_t)N)); sim->lat_cv = (int*)(lb + align_up((size_t)N) + align_up(4 * (size_t)N));
    int* scr = (int*)(lb + align_up((size_t)N) + 2 * align_up(4 * (size_t)N));      // 64 ints of scratch
    CUDA_TRY(cudaMemsetAsync(sim->lat_sub, 0xff, (size_t)N, st));
    const int nb256 = (int)((N + 255) / 256);
    int nsub = 0, rep = i0;
    for (;;) {
        if (nsub == NSUB_MAX) return lattice_fail(sim, FS_LATTICE_TOO_MANY_SUBLATTICES);
        int init[2] = {0x7fffffff, 0};
        CUDA_TRY(cudaMemcpyAsync(scr, init, sizeof(init), cudaMemcpyHostToDevice, st));
        k_lat_assign<<<nb256, 256, 0, st>>>(N, sim->lframe, rep, nsub, sim->pos, sim->cs, sim->lat_sub, sim->lat_cu,
                                            sim->lat_cv, scr); LAUNCHED();
        int res[2];
        CUDA_TRY(cudaMemcpyAsync(res, scr, sizeof(res), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        ++nsub;
        if (res[1] == 0) return lattice_fail(sim, FS_LATTICE_NOT_PERIODIC);       // representative did not match itself
        if (res[0] == 0x7fffffff) break;
        rep = res[0];
    }
    // extents
    int ext_init[8] = {0x7fffffff, 0x7fffffff, (int)0x80000000, (int)0x80000000, 0, 0, 0, 0};
    CUDA_TRY(cudaMemcpyAsync(scr, ext_init, sizeof(ext_init), cudaMemcpyHostToDevice, st));
    unsigned long long* scr64 = (unsigned long long*)(scr + 8);                   // [0] wmax, [1] dev, [2] count
    CUDA_TRY(cudaMemsetAsync(scr64, 0, 32, st));
    const int64_t NK = N * (int64_t)Kp;
    const unsigned nbk = (unsigned)((NK + 255) / 256);
    k_lat_extent<<<nbk, 256, 0, st>>>(N, Kp, sim->nbr, sim->w, sim->lat_cu, sim->lat_cv, scr, scr64); LAUNCHED();
    int ext[8]; unsigned long long wbits = 0;
    CUDA_TRY(cudaMemcpyAsync(ext, scr, sizeof(ext), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(&wbits, scr64, 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    LatGrid g{};
    g.nsub = nsub; g.u0 = ext[0]; g.v0 = ext[1];
    g.inv_nsub = (unsigned)(((1ull << 32) + nsub - 1) / nsub);
    int64_t U = (int64_t)ext[2] - ext[0] + 1, V = (int64_t)ext[3] - ext[1] + 1;
    g.Ru = ext[4]; g.Rv = ext[5];
    if (g.Ru > STENCIL_RMAX || g.Rv > STENCIL_RMAX) return lattice_fail(sim, FS_LATTICE_STENCIL_TOO_WIDE);
    int64_t Up = U + 2 * g.Ru, Vp = V + 2 * g.Rv;
    int64_t cells = (int64_t)nsub * Up * Vp;
    if (U <= 0 || V <= 0 || cells > 8 * N + (1 << 20) || Up > (1 << 30) || Vp > (1 << 30))
        return lattice_fail(sim, FS_LATTICE_TOO_SPARSE);
    g.U = (int)U; g.V = (int)V; g.Up = (int)Up; g.Vp = (int)Vp; g.W = 2 * g.Ru + 1; g.H = 2 * g.Rv + 1;
    std::memcpy(&sim->st_wmax, &wbits, 8);
    int wh = g.W * g.H;
    StencilShape shp{};
    if (!plan_stencil(sim, g, &shp)) return lattice_fail(sim, FS_LATTICE_STENCIL_TOO_WIDE);
    sim->st_nw = shp.nw; sim->st_rs = shp.rs; sim->st_pv = shp.pv; sim->st_ov = shp.ov; sim->st_smem = shp.smem;
    sim->st_ct = stencil_ct(g);
    sim->st_id = ++g_ct_next_id;
    {
        int TV = sim->st_ov * sim->st_nw;
        g.Upa = ((g.U + ST_TU - 1) / ST_TU * ST_TU + 2 * g.Ru + 3) & ~3;  // whole tiles + halo (16-byte rows): the prologue needs no bounds tests
        g.Vpa = (g.V + TV - 1) / TV * TV + 2 * g.Rv;
    }
    const size_t sg_bytes = 4 * (size_t)sim->R * nsub * g.Vpa * g.Upa;
    // tables
    size_t slots = (size_t)nsub * nsub * wh;
    size_t o_gidx = 0, o_T = align_up(4 * (size_t)cells), o_owner = o_T + align_up(16 * slots),
           o_rows = o_owner + align_up(8 * slots), o_sg = o_rows + align_up(8 * (size_t)nsub * nsub * g.W),
           o_cell = o_sg + align_up(sg_bytes), o_tf = o_cell + align_up(4 * (size_t)N), o_end = o_tf + align_up(8 * slots);
    CUDA_TRY(cudaMalloc(&sim->st_mem, o_end));
    unsigned char* sb = (unsigned char*)sim->st_mem;
    sim->gidx = (int*)(sb + o_gidx); sim->T = (double2*)(sb + o_T); sim->owner = (unsigned long long*)(sb + o_owner);
    sim->rowtab = (int2*)(sb + o_rows); sim->sgrid = (sgcell_t*)(sb + o_sg); sim->cellidx = (int*)(sb + o_cell);
    sim->Tf = (float2*)(sb + o_tf);
    CUDA_TRY(cudaMemsetAsync(sim->sgrid, 0, sg_bytes, st));
    CUDA_TRY(cudaMemsetAsync(sim->gidx, 0xff, 4 * (size_t)cells, st));
    CUDA_TRY(cudaMemsetAsync(sim->T, 0, 16 * slots, st));
    CUDA_TRY(cudaMemsetAsync(sim->owner, 0xff, 8 * slots, st));
    CUDA_TRY(cudaMemsetAsync(scr, 0, 4, st));                                      // flags
    k_lat_scatter<<<nb256, 256, 0, st>>>(N, g, sim->lat_sub, sim->lat_cu, sim->lat_cv, sim->gidx, sim->cellidx, scr); LAUNCHED();
    for (int mode = 0; mode < 3; ++mode) {
        k_stencil_build<<<nbk, 256, 0, st>>>(mode, N, Kp, g, sim->nbr, sim->w, sim->lat_sub, sim->lat_cu, sim->lat_cv,
                                             sim->owner, sim->T, scr64 + 1); LAUNCHED();
    }
    k_stencil_rows<<<(nsub * nsub * g.W + 127) / 128, 128, 0, st>>>(g, sim->owner, sim->rowtab); LAUNCHED();
    k_table_f32<<<(unsigned)((slots + 255) / 256), 256, 0, st>>>((int)slots, sim->T, sim->Tf); LAUNCHED();
    k_stencil_count<<<nb256, 256, 0, st>>>(N, g, sim->lat_sub, sim->lat_cu, sim->lat_cv, sim->gidx, sim->owner, scr64 + 2); LAUNCHED();
    int flags = 0; unsigned long long res64[3];
    CUDA_TRY(cudaMemcpyAsync(&flags, scr, 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(res64, scr64, 24, cudaMemcpyDeviceToHost, st));
    std::vector<unsigned long long> own(slots);
    CUDA_TRY(cudaMemcpyAsync(own.data(), sim->owner, 8 * slots, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    std::memcpy(&sim->st_maxdev, &res64[1], 8);
    sim->st_slots = 0;
    for (unsigned long long o : own) sim->st_slots += (o != ~0ull);
    if (flags & 4) return lattice_fail(sim, FS_LATTICE_NOT_PERIODIC);
    if ((long long)res64[2] != (long long)sim->n_inter) return lattice_fail(sim, FS_LATTICE_REACH_MISMATCH);
    // Acceptance (i): the stencil field differs from the per-pair (ELL) field by at most sum_j |w_ij - T| <= K * maxdev
    // at every spin.  On lattices with irrational coordinates (kagome: y = p * sqrt3 / 4, rounded per spin) couplings
    // of equal offsets differ by the rounding of the positions, ~3 ulp(coordinate) / d relative, so maxdev is not 0;
    // K * maxdev <= 5e-13 max|w| keeps the stencil field within 1e-12 of the per-pair field relative to max|h| for
    // every state with max|h| >= max|w| / 2.  Exact lattices (square, pinwheel) have maxdev == 0.
    if (!(sim->st_maxdev * (double)sim->K <= 5e-13 * sim->st_wmax)) return lattice_fail(sim, FS_LATTICE_WEIGHT_MISMATCH);
    const size_t stb = 200 * 1024;                       // the planner's cap: set once for every instantiation
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, true, 8, false, 64>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, true, 8, false, 64>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, false, 8, false, 64>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, false, 8, false, 64>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, true, 8, false, 128>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, true, 8, false, 128>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, false, 8, false, 128>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, false, 8, false, 128>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, true, 8, true, 64, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, true, 8, true, 64, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, true, 8, false, 64, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, true, 8, false, 64, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, true, 8, true, 128, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, true, 8, true, 128, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 7, true, 8, false, 128, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 3, true, 8, false, 128, float>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 4, true, 8, true, 64>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 2, true, 8, true, 64>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<128, 4, true, 8, true, 128>, stb));
    CUDA_TRY(raise_smem_limit(k_gather_stencil<256, 2, true, 8, true, 128>, stb));
    sim->lg = g;
    sim->st_sym = false;
    if (sim->st_ct) {
        std::vector<int2> rt((size_t)nsub * nsub * g.W);
        CUDA_TRY(cudaMemcpyAsync(rt.data(), sim->rowtab, 8 * rt.size(), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        sim->rtofs.resize(rt.size());
        for (size_t q = 0; q < rt.size(); ++q)
            sim->rtofs[q] = (int)(q / g.W) * wh + (int)(q % g.W) * g.H + (rt[q].x + g.Rv);
        int rc2 = build_inversion_pairs(sim, g, own);
        if (rc2) return rc2;
        // the paired fp64 kernel stages its tiles by TMA: without a descriptor it is not used (the plain kernel is)
        if (sim->st_sym && !make_spin_grid_map(sim, g)) sim->st_sym = false;
    }
    sim->stencil_ok = true; sim->stencil_reason = 0;
    // the build-only arrays (sub, cu, cv) are no longer needed
    cudaFree(sim->lat_mem); sim->lat_mem = nullptr; sim->lat_sub = nullptr; sim->lat_cu = sim->lat_cv = nullptr;
    return FS_OK;
}

int ensure_fields(fs_sim* sim) { return sim->fields_dirty ? do_gather(sim) : FS_OK; }

int do_scan(fs_sim* sim, bool finalize) {
    int rc = ensure_fields(sim);
    if (rc) return rc;
    const int spb = sim->LB > 512 ? 1024 : 512;
    dim3 grid((unsigned)((sim->N + spb - 1) / spb), (unsigned)sim->R);
    FieldSpec fsp{sim->sigma, sim->seed, sim->step};
#define FS_SCAN_ARGS sim->N, sim->LB, sim->ast, fsp, finalize ? 1 : 0, sim->hext, sim->cs, sim->hc, sim->s, sim->hdip, \
                     sim->hfix, sim->M, sim->bval, sim->bidx, sim->nblk, sim->scnt, sim->ctr, sim->hloc, \
                     sim->field_pending ? 1 : 0, sim->field_value
    if (spb == 1024) CUDA_TRY(launch_pdl(k_scan<2, 1024>, grid, dim3(512), 0, sim->stream, FS_SCAN_ARGS));
    else CUDA_TRY(launch_pdl(k_scan<2, 512>, grid, dim3(256), 0, sim->stream, FS_SCAN_ARGS));
    sim->field_pending = false;
#undef FS_SCAN_ARGS
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    return FS_OK;
}

int flush_field(fs_sim* sim) {
    if (!sim->field_pending) return FS_OK;
    k_set_field<<<(sim->R + 127) / 128, 128, 0, sim->stream>>>(sim->R, sim->field_value.x, sim->field_value.y, sim->hext); LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    sim->field_pending = false;
    return FS_OK;
}

int push_field(fs_sim* sim) {
    sim->field_pending = false;
    CUDA_TRY(cudaMemcpyAsync(sim->hext, sim->hext_host, sizeof(double2) * sim->R, cudaMemcpyHostToDevice, sim->stream));
    return FS_OK;
}

int fetch_counters(fs_sim* sim) {
    CUDA_TRY(cudaMemcpyAsync(sim->ctr_host, sim->ctr, sizeof(Counters) * sim->R, cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    return FS_OK;
}

// T == 0: relax at the field set by fs_set_field (k_scan first); T > 0: whole protocol in one launch
int launch_relax(fs_sim* sim, int64_t max_flips, int T, const double2* fields_dev, uint32_t step0, long long* per_step_dev,
                 const double* sigma_dev = nullptr, int use_base = 0, const double* lscale_dev = nullptr,
                 const double2* lseries_dev = nullptr) {
    int lb_shift = 0; while ((1 << lb_shift) < sim->LB) ++lb_shift;
    FieldSpec fsp{sim->sigma, sim->seed, T > 0 ? step0 : sim->step};
    // ensembles of small systems: when there are more replicas than SMs and the whole update fits one warp,
    // 128-thread CTAs (8 per SM, 64 registers) instead of 512-thread ones (1 per SM); beyond 8 replicas per
    // SM, 64-thread CTAs (16 per SM).  Measured on 220-spin replicas: 75k / 421k / 539k replica-sweeps per s.
    const bool small_cta = sim->R > sim->sm_count && sim->Kp + 1 <= 32 && sim->nblk <= 1024;
    // ensembles with more than 31 neighbours per spin (e.g. section IV.B: 592 replicas, K = 632): the loop is latency-bound,
    // so several replicas per SM beat a wide CTA per replica: 256 threads (4 per SM), 128 from 8 replicas per SM
    const bool mid_cta = sim->R > sim->sm_count && sim->Kp + 1 > 32 && sim->nblk <= 1024;
    // per-spin state in shared memory (sweeps only: a single relax would copy the state in and out for a few flips), if it
    // fits beside the hierarchy without costing the variant its CTAs per SM
    const int threads = small_cta ? (sim->R > 8 * sim->sm_count ? 64 : 128) : mid_cta ? (sim->R >= 8 * sim->sm_count ? 128 : 256)
                                  : (sim->Kp + 1 > 512 ? 1024 : 512);
    const int ctas_per_sm = threads == 64 ? 16 : threads == 128 ? 8 : threads == 256 ? 4 : 1;
    const size_t state_bytes = 49 * (size_t)sim->N + 32;
    const size_t smem_budget = std::min<size_t>(200 * 1024, (227 * 1024) / ctas_per_sm - 1024);
    const int state_smem = (T > 0 && sim->relax_smem + state_bytes <= smem_budget) ? 1 : 0;
    const size_t smem = sim->relax_smem + (state_smem ? state_bytes : 0);
#define FS_RELAX_ARGS sim->N, sim->Kp, lb_shift, sim->nblk, sim->ast, (long long)max_flips, (long long)sim->log_cap, sim->nbr, \
        sim->wT, sim->hc, sim->s, sim->hdip, sim->hfix, sim->M, sim->bval, sim->bidx, sim->flog, sim->ctr, \
        sim->stencil_ok && sim->sgrid_valid ? sim->cellidx : nullptr, sim->sgrid, \
        sim->stencil_ok ? (int64_t)sim->lg.nsub * sim->lg.Upa * sim->lg.Vpa : 0, \
        T, fields_dev, fsp, sim->cs, per_step_dev, sim->hext, sim->hloc, sigma_dev, lscale_dev, lseries_dev, use_base, state_smem
    if (threads == 64) { CUDA_TRY(raise_smem_limit(k_relax<64>, smem)); CUDA_TRY(launch_pdl(k_relax<64>, dim3((unsigned)sim->R), dim3(64), smem, sim->stream, FS_RELAX_ARGS)); }
    else if (threads == 128) { CUDA_TRY(raise_smem_limit(k_relax<128>, smem)); CUDA_TRY(launch_pdl(k_relax<128>, dim3((unsigned)sim->R), dim3(128), smem, sim->stream, FS_RELAX_ARGS)); }
    else if (threads == 256) { CUDA_TRY(raise_smem_limit(k_relax<256>, smem)); CUDA_TRY(launch_pdl(k_relax<256>, dim3((unsigned)sim->R), dim3(256), smem, sim->stream, FS_RELAX_ARGS)); }
    else if (threads == 1024) { CUDA_TRY(raise_smem_limit(k_relax<1024>, smem)); CUDA_TRY(launch_pdl(k_relax<1024>, dim3((unsigned)sim->R), dim3(1024), smem, sim->stream, FS_RELAX_ARGS)); }
    else { CUDA_TRY(raise_smem_limit(k_relax<512>, smem)); CUDA_TRY(launch_pdl(k_relax<512>, dim3((unsigned)sim->R), dim3(512), smem, sim->stream, FS_RELAX_ARGS)); }
#undef FS_RELAX_ARGS
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    return FS_OK;
}

// Exact batched flips (batch.cuh) for one large system: a cooperative kernel on all SMs commits the long prefixes of
// the flip sequence that big avalanches allow; k_relax then finishes the tail from the rebuilt leaf maxima.
int launch_batch(fs_sim* sim) {
    BatchArgs a = sim->bt;
    a.cellidx = sim->stencil_ok && sim->sgrid_valid ? sim->cellidx : nullptr;
    a.P = sim->bt_P; a.seq_threshold = sim->bt_seq; a.min_commit = sim->bt_min_commit; a.max_chain = sim->bt_max_chain;
    void* args[] = {&a};
    CUDA_TRY(cudaLaunchCooperativeKernel((const void*)k_relax_batch, dim3((unsigned)sim->bt_grid), dim3(BT_THREADS), args, 0, sim->stream));
    LAUNCHED();
    return FS_OK;
}

int do_relax(fs_sim* sim, int64_t max_flips) {
    const bool batch = sim->bt_ok && sim->bt_P > 0 && max_flips <= 0;
    int rc = do_scan(sim, batch);                        // the batched kernel wants the number of switchable spins
    if (rc) return rc;
    if (batch) { rc = launch_batch(sim); if (rc) return rc; }
    return launch_relax(sim, max_flips, 0, nullptr, 0, nullptr, nullptr, batch ? 1 : 0);
}

// scratch of k_relax_batch; never fails the creation (no scratch = sequential relax only)
int setup_batch(fs_sim* sim) {
    sim->bt_ok = false;
    if (!batch_applies(sim->N, sim->R, sim->K) || !sim->bt_mem) return FS_OK;
    int coop = 0, occ = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, sim->device);
    if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_relax_batch, BT_THREADS, 0) != cudaSuccess || occ < 1) {
        cudaGetLastError(); return FS_OK;
    }
    const BatchLayout bl = batch_layout(sim->N, sim->K, sim->Kp);
    const int Pdef = bl.Pdef, P = bl.P;
    const size_t o_ctl = bl.ctl, o_owner = bl.owner, o_seeds = bl.seeds, o_edges = bl.edges, o_ecount = bl.ecount,
                 o_npos = bl.npos, o_elems = bl.elems, o_undo = bl.undo, o_blocks = bl.blocks, o_clist = bl.clist,
                 o_cand = bl.cand, o_cbits = bl.cbits;
    unsigned char* b = (unsigned char*)sim->bt_mem;      // the workspace's batch region (fs_create laid it out)
    int lb_shift = 0; while ((1 << lb_shift) < sim->LB) ++lb_shift;
    BatchArgs& a = sim->bt;
    a.N = sim->N; a.Kp = sim->Kp; a.LBshift = lb_shift; a.nblk = sim->nblk; a.ast = sim->ast; a.log_cap = sim->log_cap;
    a.nbr = sim->nbr; a.wT = sim->wT; a.ihc = sim->hc; a.s = sim->s; a.hdip = sim->hdip; a.hfix = sim->hfix; a.M = sim->M;
    a.bval = sim->bval; a.bidx = sim->bidx; a.flog = sim->flog; a.ctr = sim->ctr;
    a.cellidx = nullptr; a.sgrid = sim->sgrid;
    a.ctl = (BatchCtl*)(b + o_ctl); a.owner = (unsigned*)(b + o_owner); a.seeds = (BatchSeed*)(b + o_seeds);
    a.edges = (unsigned short*)(b + o_edges); a.ecount = b + o_ecount; a.npos = (int*)(b + o_npos);
    a.elems = (BatchElem*)(b + o_elems); a.undo = (BatchUndo*)(b + o_undo); a.blocks = (BatchBlock*)(b + o_blocks);
    a.clist = (BatchCommit*)(b + o_clist); a.cand = (int*)(b + o_cand); a.cbits = (unsigned*)(b + o_cbits);
    if (cudaMemsetAsync(a.ctl, 0, sizeof(BatchCtl), sim->stream) != cudaSuccess ||
        cudaMemsetAsync(a.owner, 0xff, 4 * (size_t)sim->N, sim->stream) != cudaSuccess) {
        cudaGetLastError(); return FS_OK;
    }
    sim->bt_P = Pdef; sim->bt_alloc = P; sim->bt_seq = 64; sim->bt_grid = sim->sm_count; sim->bt_ok = true;
    return FS_OK;
}

}  // namespace

extern "C" {

const char* fs_last_error(void) { return g_err; }
int64_t fs_kernel_launches(void) { return (int64_t)g_launches.load(); }

int fs_workspace_bytes(int64_t N, int32_t R, const double* pos_dev, const fs_params* p, size_t* bytes_out, void* stream) {
    int rc = check_params(N, R, p);
    if (rc) return rc;
    if (!pos_dev || !bytes_out) return fail(FS_ERR_ARG, "null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    double* bbox = nullptr;
    CUDA_TRY(cudaMalloc(&bbox, 256));
    GridPlan gp;
    rc = plan_grid(N, pos_dev, p, bbox, st, &gp);
    cudaFree(bbox);
    if (rc) return rc;
    Layout L{};
    layout_grid(L, N, gp.ncells);
    unsigned char* tmp = nullptr;
    CUDA_TRY(cudaMalloc(&tmp, L.grid_end));
    cudaMemsetAsync(tmp, 0, 256, st);
    int K = 0, flags = 0; long long I = 0;
    rc = build_grid_and_count(N, pos_dev, gp, tmp, L, st, &K, &I, &flags);
    cudaFree(tmp);
    if (rc) return rc;
    if (flags & 2) return fail(FS_ERR_COINCIDENT, "two spins share a position");
    if (K > MAX_K) return fail(FS_ERR_ARG, "max degree %d exceeds %d", K, MAX_K);
    int LB, nblk;
    if (choose_leaf(N, &LB, &nblk)) return fail(FS_ERR_ARG, "N too large for the relax hierarchy");
    layout_rest(L, N, R, K, pad_k(K), nblk, 4 * N + 1024);
    *bytes_out = L.total;
    return FS_OK;
}

int fs_create_ensemble(fs_sim** out, int64_t N, int32_t R, const double* pos_dev, const double* angle_dev,
                       const double* hc_dev, const fs_params* p, void* workspace_dev, size_t workspace_bytes,
                       void* stream) {
    int rc = check_params(N, R, p);
    if (rc) return rc;
    if (!out || !pos_dev || !angle_dev || !hc_dev || !workspace_dev) return fail(FS_ERR_ARG, "null pointer");
    if (((uintptr_t)workspace_dev & 255u) != 0) return fail(FS_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char* base = (unsigned char*)workspace_dev;
    if (workspace_bytes < 256) return fail(FS_ERR_WORKSPACE, "workspace too small");
    CUDA_TRY(cudaMemsetAsync(base, 0, 256, st));

    GridPlan gp;
    rc = plan_grid(N, pos_dev, p, (double*)base, st, &gp);
    if (rc) return rc;
    Layout L{};
    layout_grid(L, N, gp.ncells);
    if (workspace_bytes < L.grid_end) return fail(FS_ERR_WORKSPACE, "workspace too small (%zu < %zu)", workspace_bytes, L.grid_end);
    int K = 0, flags = 0; long long I = 0;
    rc = build_grid_and_count(N, pos_dev, gp, base, L, st, &K, &I, &flags);
    if (rc) return rc;
    if (flags & 2) return fail(FS_ERR_COINCIDENT, "two spins share a position");
    if (K > MAX_K) return fail(FS_ERR_ARG, "max degree %d exceeds %d", K, MAX_K);
    int LB, nblk;
    if (choose_leaf(N, &LB, &nblk)) return fail(FS_ERR_ARG, "N too large for the relax hierarchy");
    int Kp = pad_k(K);
    int64_t log_cap = 4 * N + 1024;
    layout_rest(L, N, R, K, Kp, nblk, log_cap);
    if (workspace_bytes < L.total) return fail(FS_ERR_WORKSPACE, "workspace too small (%zu < %zu)", workspace_bytes, L.total);

    fs_sim* sim = new (std::nothrow) fs_sim();
    if (!sim) return fail(FS_ERR_ARG, "out of host memory");
    sim->N = N; sim->R = R; sim->K = K; sim->Kp = Kp; sim->LB = LB; sim->nblk = nblk; sim->ncells = gp.ncells;
    sim->n_inter = I; sim->log_cap = log_cap; sim->p = *p; sim->grid = gp.g; sim->stream = st;
    auto kind = [](double denom) { return denom == 3.0 ? 1 : (denom == 2.0 ? 2 : (denom == 1.0 ? 3 : 0)); };
    sim->ast = Astroid{1.0 / p->b, 1.0 / p->c, 2.0 / p->gamma, 2.0 / p->beta, kind(p->gamma), kind(p->beta),
                       std::pow(0.5, p->gamma / 2.0) * (1.0 - 1e-9), std::pow(0.5, p->beta / 2.0) * (1.0 - 1e-9)};
    int dev = 0; cudaGetDevice(&dev);
    sim->device = dev;
    cudaDeviceGetAttribute(&sim->sm_count, cudaDevAttrMultiProcessorCount, dev);
    sim->pos = (double2*)(base + L.pos); sim->cs = (double2*)(base + L.cs);
    sim->nbr = (int*)(base + L.nbr); sim->w = (double2*)(base + L.w); sim->wT = (double2*)(base + L.wT);
    sim->deg = (int*)(base + L.deg);
    sim->hc = (double*)(base + L.hc); sim->s = (int8_t*)(base + L.s);
    sim->hdip = (double2*)(base + L.hdip); sim->hfix = (double2*)(base + L.hfix); sim->M = (double*)(base + L.M);
    sim->bval = (double*)(base + L.bval); sim->bidx = (int*)(base + L.bidx); sim->flog = (int*)(base + L.flog);
    sim->scnt = (unsigned*)(base + L.scnt);
    sim->ctr = (Counters*)(base + L.ctr); sim->hext = (double2*)(base + L.hext);
    sim->hloc_buf = (double2*)(base + L.hloc);
    sim->bt_mem = batch_applies(N, R, K) ? (void*)(base + L.batch) : nullptr;

#define CREATE_TRY(expr)                                                                           \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            fs_destroy(sim);                                                                       \
            return fail(FS_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
        }                                                                                          \
    } while (0)
    CREATE_TRY(cudaMallocHost(&sim->hext_host, sizeof(double2) * R));
    CREATE_TRY(cudaMallocHost(&sim->ctr_host, sizeof(Counters) * R));
    for (int r = 0; r < R; ++r) sim->hext_host[r] = make_double2(0.0, 0.0);

    CREATE_TRY(cudaMemcpyAsync(sim->pos, pos_dev, 16 * (size_t)N, cudaMemcpyDeviceToDevice, st));
    CREATE_TRY(cudaMemcpyAsync(sim->hc, hc_dev, 8 * (size_t)R * N, cudaMemcpyDeviceToDevice, st));
    CREATE_TRY(cudaMemsetAsync(sim->ctr, 0, sizeof(Counters) * R, st));
    CREATE_TRY(cudaMemsetAsync(sim->scnt, 0, 4 * (size_t)R * scan_aux_stride((int)((N + SCAN_SPB_MIN - 1) / SCAN_SPB_MIN)), st));
    CREATE_TRY(cudaMemsetAsync(sim->hdip, 0, 16 * (size_t)R * N, st));
    CREATE_TRY(cudaMemcpyAsync(sim->hext, sim->hext_host, sizeof(double2) * R, cudaMemcpyHostToDevice, st));
    int nb = (int)((N + 255) / 256);
    int* scr = (int*)(base + L.scratch);
    k_frame<<<nb, 256, 0, st>>>(N, R, angle_dev, sim->hc, sim->cs, scr + 8); LAUNCHED();
    {
        int64_t rn = (int64_t)R * N;
        k_fill_i8<<<(unsigned)((rn + 255) / 256), 256, 0, st>>>(rn, (int8_t)1, sim->s); LAUNCHED();
    }
    // A1 fill + sort
    int Kp2 = 2; while (Kp2 < Kp) Kp2 <<= 1;
    {
        int warps = 4;
        size_t smem = (size_t)warps * Kp2 * sizeof(int);
        CREATE_TRY(raise_smem_limit(k_fill_neighbors, smem));
        int64_t blocks = std::min<int64_t>((N + warps - 1) / warps, (int64_t)sim->sm_count * 16);
        k_fill_neighbors<<<(unsigned)blocks, warps * 32, smem, st>>>(N, gp.g, gp.cut2, Kp, Kp2, sim->pos,
                                                                      (int*)(base + L.cell_start), (int*)(base + L.items), sim->nbr);
        LAUNCHED();
    }
    // A2 weights
    {
        int64_t tot = N * (int64_t)Kp;
        k_weights<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(N, Kp, p->alpha, sim->pos, sim->cs, sim->nbr, sim->w, sim->wT);
        LAUNCHED();
    }
    sim->relax_smem = ((size_t)nblk + (size_t)(nblk + 31) / 32 + 8) * 12 + (size_t)(Kp + 1) * 4 + 32;
    CREATE_TRY(raise_smem_limit(k_relax<512>, sim->relax_smem));
    CREATE_TRY(raise_smem_limit(k_relax<128>, sim->relax_smem));
    CREATE_TRY(raise_smem_limit(k_relax<256>, sim->relax_smem));
    CREATE_TRY(raise_smem_limit(k_relax<64>, sim->relax_smem));
    CREATE_TRY(raise_smem_limit(k_relax<1024>, sim->relax_smem));
    int hflags = 0;
    CREATE_TRY(cudaMemcpyAsync(&hflags, scr + 8, sizeof(int), cudaMemcpyDeviceToHost, st));
    CREATE_TRY(cudaStreamSynchronize(st));
    CREATE_TRY(cudaGetLastError());
#undef CREATE_TRY
    if (hflags & 1) { fs_destroy(sim); return fail(FS_ERR_ARG, "hc must be finite and > 0, angle finite"); }
    rc = detect_lattice(sim);
    if (rc) { fs_destroy(sim); return rc; }
    setup_batch(sim);
    sim->fields_dirty = true;
    *out = sim;
    return FS_OK;
}

int fs_create(fs_sim** out, int64_t N, const double* pos_dev, const double* angle_dev, const double* hc_dev,
              const fs_params* p, void* workspace_dev, size_t workspace_bytes, void* stream) {
    return fs_create_ensemble(out, N, 1, pos_dev, angle_dev, hc_dev, p, workspace_dev, workspace_bytes, stream);
}

int fs_destroy(fs_sim* sim) {
    if (!sim) return FS_OK;
    DeviceGuard guard_(sim->device);
    cudaStreamSynchronize(sim->stream);                  // kernels in flight may still read the pinned staging buffers
    if (sim->hext_host) cudaFreeHost(sim->hext_host);
    if (sim->ctr_host) cudaFreeHost(sim->ctr_host);
    if (sim->lat_mem) cudaFree(sim->lat_mem);
    if (sim->st_mem) cudaFree(sim->st_mem);
    delete sim;
    return FS_OK;
}

int fs_get_info(const fs_sim* sim, int64_t* N, int32_t* R, int32_t* K, int64_t* n_interactions) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (N) *N = sim->N;
    if (R) *R = sim->R;
    if (K) *K = sim->K;
    if (n_interactions) *n_interactions = sim->n_inter;
    return FS_OK;
}

int fs_set_spins(fs_sim* sim, const int8_t* s_dev) {
    if (!sim || !s_dev) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    CUDA_TRY(cudaMemcpyAsync(sim->s, s_dev, (size_t)sim->R * sim->N, cudaMemcpyDeviceToDevice, sim->stream));
    sim->fields_dirty = true; sim->sgrid_valid = false;
    return FS_OK;
}

int fs_get_spins(fs_sim* sim, int8_t* s_dev_out) {
    if (!sim || !s_dev_out) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    CUDA_TRY(cudaMemcpyAsync(s_dev_out, sim->s, (size_t)sim->R * sim->N, cudaMemcpyDeviceToDevice, sim->stream));
    return FS_OK;
}

int fs_set_thermal(fs_sim* sim, double sigma_th, uint64_t seed) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (!(sigma_th >= 0.0)) return fail(FS_ERR_ARG, "sigma_th must be >= 0");
    sim->sigma = sigma_th; sim->seed = seed;
    return FS_OK;
}

int fs_set_field(fs_sim* sim, double hx, double hy, uint32_t step) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    sim->step = step;
    // no launch and no host sync: the next scan takes the value as a kernel argument (one launch less per field step);
    // the few other readers of sim->hext call flush_field first
    sim->field_pending = true; sim->field_value = make_double2(hx, hy);
    return FS_OK;
}

int fs_set_field_ensemble(fs_sim* sim, const double* h_host, uint32_t step) {
    if (!sim || !h_host) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    for (int r = 0; r < sim->R; ++r) sim->hext_host[r] = make_double2(h_host[2 * r], h_host[2 * r + 1]);
    sim->step = step;
    return push_field(sim);
}

int fs_set_local_field(fs_sim* sim, const double* h_dev) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (!h_dev) { sim->hloc = nullptr; return FS_OK; }   // kernels already enqueued keep reading the workspace copy
    sim->hloc = sim->hloc_buf;
    CUDA_TRY(cudaMemcpyAsync(sim->hloc, h_dev, 16 * (size_t)sim->N, cudaMemcpyDeviceToDevice, sim->stream));
    return FS_OK;
}

int fs_set_gather_variant(fs_sim* sim, int variant) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (variant < 0 || variant > 4) return fail(FS_ERR_ARG, "unknown gather variant %d", variant);
    if (variant == FS_GATHER_STENCIL_F32 && !(sim->stencil_ok && sim->st_ct))
        return fail(FS_ERR_ARG, "fp32 stencil gather unavailable (needs a verified lattice whose table fits constant memory)");
    if ((variant == FS_GATHER_STENCIL || variant == FS_GATHER_STENCIL_PLAIN) && !sim->stencil_ok)
        return fail(FS_ERR_ARG, "stencil gather unavailable for this geometry (FS_LATTICE reason %d)", sim->stencil_reason);
    sim->gather_variant = variant;
    return FS_OK;
}

int fs_get_lattice(const fs_sim* sim, int32_t* info, double* dinfo) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (info) {
        const LatGrid& g = sim->lg;
        int32_t v[12] = {sim->stencil_ok ? 1 : 0, sim->stencil_reason, g.nsub, g.U, g.V, g.Ru, g.Rv,
                         (int32_t)sim->st_slots, sim->st_nw * sim->st_rs, (int32_t)sim->st_smem,
                         sim->stencil_ok && sim->st_sym ? 1 : 0, (int32_t)sim->prow.size()};
        for (int k = 0; k < 12; ++k) info[k] = v[k];
    }
    if (dinfo) { dinfo[0] = sim->st_maxdev; dinfo[1] = sim->st_wmax; }
    return FS_OK;
}

int fs_measure_fp64_peak(double* dfma_per_s, void* stream) {
    if (!dfma_per_s) return fail(FS_ERR_ARG, "null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    CUDA_TRY(cudaMalloc(&sink, 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 1 << 14, blocks = sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        k_dfma_peak<<<blocks, threads, 0, st>>>(iters, 1.0 + rep, sink); LAUNCHED();
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        double rate = 8.0 * iters * (double)blocks * threads / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    CUDA_TRY(cudaGetLastError());
    *dfma_per_s = best;
    return FS_OK;
}

int fs_measure_fp32_peak(double* ffma_per_s, void* stream) {
    if (!ffma_per_s) return fail(FS_ERR_ARG, "null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* sink = nullptr;
    CUDA_TRY(cudaMalloc(&sink, 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 1 << 15, blocks = sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        k_ffma_peak<<<blocks, threads, 0, st>>>(iters, 1.0f + rep, sink); LAUNCHED();
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        double rate = 8.0 * iters * (double)blocks * threads / (ms * 1e-3);
        if (rep > 0 && rate > best) best = rate;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    CUDA_TRY(cudaGetLastError());
    *ffma_per_s = best;
    return FS_OK;
}

#ifdef FS_BATCH_PROFILE
int fs_debug_batch_profile(fs_sim* sim, long long* out12) {
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpy(out12, sim->bt.ctl->prof, sizeof(long long) * 12, cudaMemcpyDeviceToHost));
    return FS_OK;
}
#endif

#ifdef FS_RELAX_PROFILE
int fs_debug_relax_profile(long long* out16, int reset) {
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpyFromSymbol(out16, g_relax_prof, sizeof(long long) * 16));
    if (reset) { long long z[16] = {0}; CUDA_TRY(cudaMemcpyToSymbol(g_relax_prof, z, sizeof(z))); }
    return FS_OK;
}
#endif

int fs_set_batch(fs_sim* sim, int32_t max_seeds, int32_t seq_threshold) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    if (max_seeds < 0 || max_seeds > BT_PMAX || seq_threshold < 0) return fail(FS_ERR_ARG, "max_seeds must be in [0, %d], seq_threshold >= 0", BT_PMAX);
    if (max_seeds > 0 && !sim->bt_ok) return fail(FS_ERR_ARG, "batched flips unavailable for this simulation (needs R = 1, 1 <= K <= 64, N >= 16384)");
    if (sim->bt_ok) {
        sim->bt_P = std::min<int>(max_seeds, sim->bt_alloc);
        sim->bt_seq = seq_threshold;
    }
    return FS_OK;
}

int fs_get_batch_stats(fs_sim* sim, int64_t* out4) {
    if (!sim || !out4) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    int rc = fetch_counters(sim);
    if (rc) return rc;
    out4[0] = sim->bt_ok ? sim->bt_P : 0;
    out4[1] = sim->ctr_host[0].batch_total;
    out4[2] = sim->ctr_host[0].batch_rounds;
    out4[3] = sim->bt_seq;
    return FS_OK;
}

int fs_update_fields(fs_sim* sim) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    return do_gather(sim);
}

int fs_scan_ensemble(fs_sim* sim, int64_t* n_switchable, int64_t* best_index, double* best_L) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    int rc = do_scan(sim, true);
    if (rc) return rc;
    if (!n_switchable && !best_index && !best_L) return FS_OK;
    rc = fetch_counters(sim);
    if (rc) return rc;
    for (int r = 0; r < sim->R; ++r) {
        if (n_switchable) n_switchable[r] = sim->ctr_host[r].n_switchable;
        if (best_index) best_index[r] = sim->ctr_host[r].best_index;
        if (best_L) best_L[r] = sim->ctr_host[r].best_L;
    }
    return FS_OK;
}

int fs_scan(fs_sim* sim, int64_t* n_switchable, int64_t* best_index, double* best_L) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (sim->R == 1) return fs_scan_ensemble(sim, n_switchable, best_index, best_L);
    int rc = fs_scan_ensemble(sim, nullptr, nullptr, nullptr);
    if (rc) return rc;
    if (!n_switchable && !best_index && !best_L) return FS_OK;
    rc = fetch_counters(sim);
    if (rc) return rc;
    if (n_switchable) *n_switchable = sim->ctr_host[0].n_switchable;
    if (best_index) *best_index = sim->ctr_host[0].best_index;
    if (best_L) *best_L = sim->ctr_host[0].best_L;
    return FS_OK;
}

int fs_relax_ensemble(fs_sim* sim, int64_t max_flips, int64_t* n_flips_out) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    int rc = do_relax(sim, max_flips);
    if (rc) return rc;
    if (!n_flips_out) return FS_OK;
    rc = fetch_counters(sim);
    if (rc) return rc;
    int capped = 0;
    for (int r = 0; r < sim->R; ++r) { n_flips_out[r] = sim->ctr_host[r].last_flips; capped |= sim->ctr_host[r].status; }
    return capped ? fail(FS_ERR_MAXFLIPS, "relax stopped at max_flips=%lld", (long long)max_flips) : FS_OK;
}

int fs_relax(fs_sim* sim, int64_t max_flips, int64_t* n_flips_out) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    int rc = do_relax(sim, max_flips);
    if (rc) return rc;
    if (!n_flips_out) return FS_OK;
    rc = fetch_counters(sim);
    if (rc) return rc;
    int64_t tot = 0; int capped = 0;
    for (int r = 0; r < sim->R; ++r) { tot += sim->ctr_host[r].last_flips; capped |= sim->ctr_host[r].status; }
    *n_flips_out = tot;
    return capped ? fail(FS_ERR_MAXFLIPS, "relax stopped at max_flips=%lld", (long long)max_flips) : FS_OK;
}

int fs_sweep_ex(fs_sim* sim, const double* fields_dev, const double* sigma_dev, const double* local_scale_dev,
                const double* local_series_dev, int32_t T, uint32_t step0, int64_t* flips_per_step_dev, int64_t max_flips,
                int64_t* n_flips_out) {
    if (!sim || !fields_dev) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    if (T <= 0) return fail(FS_ERR_ARG, "T=%d must be positive", (int)T);
    int rc = ensure_fields(sim);
    if (rc) return rc;
    rc = launch_relax(sim, max_flips, T, reinterpret_cast<const double2*>(fields_dev), step0,
                      reinterpret_cast<long long*>(flips_per_step_dev), sigma_dev, 0, local_scale_dev,
                      reinterpret_cast<const double2*>(local_series_dev));
    if (rc) return rc;
    sim->step = step0 + (uint32_t)(T - 1);
    sim->field_pending = false;                          // the sweep left its own last field in sim->hext
    if (!n_flips_out) return FS_OK;
    rc = fetch_counters(sim);
    if (rc) return rc;
    int capped = 0;
    for (int r = 0; r < sim->R; ++r) { n_flips_out[r] = sim->ctr_host[r].last_flips; capped |= sim->ctr_host[r].status; }
    if (capped) sim->step = step0 + (uint32_t)sim->ctr_host[0].last_step;      // replica 0's last step (see flatspin.h)
    return capped ? fail(FS_ERR_MAXFLIPS, "sweep stopped at max_flips=%lld", (long long)max_flips) : FS_OK;
}

int fs_sweep_anneal(fs_sim* sim, const double* fields_dev, const double* sigma_dev, int32_t T, uint32_t step0,
                    int64_t* flips_per_step_dev, int64_t max_flips, int64_t* n_flips_out) {
    return fs_sweep_ex(sim, fields_dev, sigma_dev, nullptr, nullptr, T, step0, flips_per_step_dev, max_flips, n_flips_out);
}

int fs_sweep(fs_sim* sim, const double* fields_dev, int32_t T, uint32_t step0, int64_t* flips_per_step_dev,
             int64_t max_flips, int64_t* n_flips_out) {
    return fs_sweep_anneal(sim, fields_dev, nullptr, T, step0, flips_per_step_dev, max_flips, n_flips_out);
}

int fs_get_counters(fs_sim* sim, int64_t* total_flips, int64_t* last_relax_flips, int reset) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    int rc = fetch_counters(sim);
    if (rc) return rc;
    for (int r = 0; r < sim->R; ++r) {
        if (total_flips) total_flips[r] = sim->ctr_host[r].total_flips;
        if (last_relax_flips) last_relax_flips[r] = sim->ctr_host[r].last_flips;
    }
    if (reset) CUDA_TRY(cudaMemsetAsync(sim->ctr, 0, sizeof(Counters) * sim->R, sim->stream));
    return FS_OK;
}

int fs_get_fields(fs_sim* sim, int which, double* h_dev_out) {
    if (!sim || !h_dev_out) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    if (which < 0 || which > 3) return fail(FS_ERR_ARG, "unknown field selector %d", which);
    if (which == FS_FIELD_TOTAL || which == FS_FIELD_DIP) { int rc = ensure_fields(sim); if (rc) return rc; }
    { int rc = flush_field(sim); if (rc) return rc; }
    dim3 grid((unsigned)((sim->N + 255) / 256), (unsigned)sim->R);
    FieldSpec fsp{sim->sigma, sim->seed, sim->step};
    k_fields_out<<<grid, 256, 0, sim->stream>>>(sim->N, which, fsp, sim->hext, sim->cs, sim->hdip, (double2*)h_dev_out, sim->hloc);
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    return FS_OK;
}

int fs_get_flip_log_window(fs_sim* sim, int32_t replica, int32_t* idx_dev_out, int64_t cap, int64_t* n_out, int64_t* first_out) {
    if (!sim || !n_out) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    if (replica < 0 || replica >= sim->R) return fail(FS_ERR_ARG, "replica out of range");
    int rc = fetch_counters(sim);
    if (rc) return rc;
    const int64_t n = sim->ctr_host[replica].last_flips, L = sim->log_cap;
    const int64_t first = std::max<int64_t>(0, n - L);           // oldest flip still in the ring
    *n_out = n;
    if (first_out) *first_out = first;
    const int64_t ncopy = std::min(cap, n - first);
    if (ncopy > 0) {
        if (!idx_dev_out) return fail(FS_ERR_ARG, "null output buffer");
        const int32_t* base = sim->flog + (int64_t)replica * L;
        const int64_t p0 = first % L, n1 = std::min(ncopy, L - p0);          // flip number q sits at q % L
        CUDA_TRY(cudaMemcpyAsync(idx_dev_out, base + p0, 4 * (size_t)n1, cudaMemcpyDeviceToDevice, sim->stream));
        if (ncopy > n1)
            CUDA_TRY(cudaMemcpyAsync(idx_dev_out + n1, base, 4 * (size_t)(ncopy - n1), cudaMemcpyDeviceToDevice, sim->stream));
    }
    return FS_OK;
}

int fs_get_flip_log(fs_sim* sim, int32_t replica, int32_t* idx_dev_out, int64_t cap, int64_t* n_out) {
    return fs_get_flip_log_window(sim, replica, idx_dev_out, cap, n_out, nullptr);
}

int fs_get_neighbors(fs_sim* sim, int32_t* idx_dev_out, int32_t* K_out) {
    if (!sim) return fail(FS_ERR_ARG, "sim is NULL");
    DeviceGuard guard_(sim->device);
    if (K_out) *K_out = sim->K;
    if (idx_dev_out && sim->K > 0)
        CUDA_TRY(cudaMemcpy2DAsync(idx_dev_out, 4 * (size_t)sim->K, sim->nbr, 4 * (size_t)sim->Kp, 4 * (size_t)sim->K,
                                   (size_t)sim->N, cudaMemcpyDeviceToDevice, sim->stream));
    return FS_OK;
}

int fs_correlation(fs_sim* sim, double bin_width, int32_t nbins, int64_t* sum_dev, int64_t* count_dev) {
    if (!sim || !sum_dev || !count_dev) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    if (!(bin_width > 0.0) || nbins <= 0 || nbins > CORR_MAX_BINS) return fail(FS_ERR_ARG, "bin_width must be > 0 and 0 < nbins <= %d", CORR_MAX_BINS);
    CUDA_TRY(cudaMemsetAsync(sum_dev, 0, 8 * (size_t)sim->R * nbins, sim->stream));
    CUDA_TRY(cudaMemsetAsync(count_dev, 0, 8 * (size_t)nbins, sim->stream));
    if (sim->K == 0) return FS_OK;
    const int64_t total = sim->N * (int64_t)sim->Kp;
    const unsigned nb = (unsigned)std::min<int64_t>((total + 255) / 256, (int64_t)sim->sm_count * 8);
    k_correlation<<<dim3(nb, (unsigned)sim->R), 256, 0, sim->stream>>>(sim->N, sim->Kp, bin_width, nbins, sim->pos, sim->cs, sim->nbr,
                                                                          sim->s, (long long*)sum_dev, (long long*)count_dev);
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    return FS_OK;
}

int fs_vertex_populations(fs_sim* sim, const int32_t* vertices_dev, int64_t V, int64_t* counts_dev) {
    if (!sim || !counts_dev || (V > 0 && !vertices_dev)) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    if (V < 0) return fail(FS_ERR_ARG, "V must be >= 0");
    CUDA_TRY(cudaMemsetAsync(counts_dev, 0, 8 * (size_t)sim->R * 4, sim->stream));
    if (V == 0) return FS_OK;
    const unsigned nb = (unsigned)std::min<int64_t>((V + 255) / 256, (int64_t)sim->sm_count * 8);
    k_vertex_populations<<<dim3(nb, (unsigned)sim->R), 256, 0, sim->stream>>>(sim->N, V, vertices_dev, sim->pos, sim->cs, sim->s,
                                                                                 (long long*)counts_dev);
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    return FS_OK;
}

int fs_step_host(fs_sim* sim, const int8_t* s_host, double* h_host_out, int64_t* n_switchable, int64_t* best_index,
                 double* best_L) {
    if (!sim || !s_host) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    size_t rn = (size_t)sim->R * sim->N;
    CUDA_TRY(cudaMemcpyAsync(sim->s, s_host, rn, cudaMemcpyHostToDevice, sim->stream));
    sim->fields_dirty = true; sim->sgrid_valid = false;
    int rc = do_gather(sim);
    if (rc) return rc;
    rc = fs_scan_ensemble(sim, nullptr, nullptr, nullptr);
    if (rc) return rc;
    if (h_host_out) {                                    // NULL: only the scan's summary goes back to the host
        // total field into hfix's sibling buffer M is not large enough; reuse hfix (rewritten by the next scan)
        dim3 grid((unsigned)((sim->N + 255) / 256), (unsigned)sim->R);
        FieldSpec fsp{sim->sigma, sim->seed, sim->step};
        k_fields_out<<<grid, 256, 0, sim->stream>>>(sim->N, FS_FIELD_TOTAL, fsp, sim->hext, sim->cs, sim->hdip, sim->hfix, sim->hloc);
        LAUNCHED();
        CUDA_TRY(cudaMemcpyAsync(h_host_out, sim->hfix, 16 * rn, cudaMemcpyDeviceToHost, sim->stream));
    }
    rc = fetch_counters(sim);
    if (rc) return rc;
    if (n_switchable) *n_switchable = sim->ctr_host[0].n_switchable;
    if (best_index) *best_index = sim->ctr_host[0].best_index;
    if (best_L) *best_L = sim->ctr_host[0].best_L;
    return FS_OK;
}

int fs_relax_host(fs_sim* sim, double hx, double hy, uint32_t step, int8_t* s_host_out, int64_t* n_flips_out) {
    if (!sim || !s_host_out) return fail(FS_ERR_ARG, "null pointer");
    DeviceGuard guard_(sim->device);
    int rc = fs_set_field(sim, hx, hy, step);
    if (rc) return rc;
    rc = do_relax(sim, 0);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(s_host_out, sim->s, (size_t)sim->R * sim->N, cudaMemcpyDeviceToHost, sim->stream));
    rc = fetch_counters(sim);
    if (rc) return rc;
    if (n_flips_out) {
        int64_t tot = 0;
        for (int r = 0; r < sim->R; ++r) tot += sim->ctr_host[r].last_flips;
        *n_flips_out = tot;
    }
    return FS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// fs_scan_static: the switching scan (A4-A7) for callers that must not allocate device memory.
//
// Who needs it.  A host program that has handed (nearly) all of the GPU's memory to its own pool (a torch caching
// allocator sized for the 11.5 GB config-5 workspace, a solver that reserves the card at start-up) cannot let a
// library call cudaMalloc behind its back: the call fails, or it takes memory the pool counts on.  A program that keeps
// several streams busy (one ensemble member per stream) cannot afford it either: cudaMalloc and cudaFree synchronise
// the whole device.  Every other scan in this file works on a simulation handle, whose per-CTA partial results live
// in the workspace that fs_create laid out; this entry point has no handle and no workspace.  Its partial results go
// to the file-scope array below, which the CUDA module carries: FS_SCAN_STATIC_SCRATCH_BYTES (65,792 B) on every
// device that loads the library, until the process exits.  The caller passes the inputs and the 24-byte result.
//
// The arithmetic is k_scan's, through the same device functions (sincos for the frame, 1 / h_c, fixed_field, margin,
// warp_argmax_margin), so the result is the one fs_scan gives for the same h_dip.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int SCAN_STATIC_SPB = 1024;                                   // spins per CTA: 256 threads x 4 spins
constexpr int SCAN_STATIC_THREADS = 256;
constexpr int SCAN_STATIC_MAX_CTAS = FS_SCAN_STATIC_MAX_N / SCAN_STATIC_SPB;
constexpr size_t SCAN_STATIC_HEADER = 256;                              // word 0: the ticket counter; must be 0 at launch
static_assert(SCAN_STATIC_HEADER + sizeof(ScanGroup) * SCAN_STATIC_MAX_CTAS == FS_SCAN_STATIC_SCRATCH_BYTES,
              "flatspin.h states the size of the static scratch array");

// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address, and a kernel handed
// `g_scan_static_scratch` itself would read host memory or fault.  static_scratch_of() below asks the runtime for the
// address on the current device and the entry point passes that to the kernel.
static __device__ __align__(256) unsigned char g_scan_static_scratch[FS_SCAN_STATIC_SCRATCH_BYTES];

__global__ void __launch_bounds__(SCAN_STATIC_THREADS)
k_scan_static(int64_t N, Astroid ast, FieldSpec fs, double2 he, const double* __restrict__ angle,
              const double* __restrict__ hc, const int8_t* __restrict__ s, const double2* __restrict__ hdip,
              unsigned char* __restrict__ scratch, long long* __restrict__ result) {
    __shared__ double wv[SCAN_STATIC_SPB / 32];           // arg-max of every 32-spin slot of this CTA
    __shared__ int wi[SCAN_STATIC_SPB / 32];
    __shared__ unsigned wcnt[SCAN_STATIC_THREADS / 32];
    __shared__ unsigned long long wc[SCAN_STATIC_THREADS / 32];
    __shared__ int is_last;
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    ScanGroup* cres = reinterpret_cast<ScanGroup*>(scratch + SCAN_STATIC_HEADER);      // [gridDim.x]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int64_t base = (int64_t)blockIdx.x * SCAN_STATIC_SPB + threadIdx.x;
    unsigned nsw = 0;
#pragma unroll
    for (int q = 0; q < SCAN_STATIC_SPB / SCAN_STATIC_THREADS; ++q) {
        const int64_t i = base + q * SCAN_STATIC_THREADS;
        double m = -CUDART_INF; int mi = 0x7fffffff;
        if (i < N) {
            double sn, c;
            sincos(angle[i], &sn, &c);                     // k_frame's table entry (Eq. 1)
            const double ih = 1.0 / hc[i];
            const double2 hd = hdip[i];
            const double2 hf = fixed_field(make_double2(c, sn), he, fs, 0, (uint32_t)i);
            m = margin(hd.x + hf.x, hd.y + hf.y, (double)s[i], ih, ast);
            mi = (int)i;
        }
        nsw += __popc(__ballot_sync(0xffffffffu, m > 1.0));
        warp_argmax_margin(m, mi);
        if (lane == 0) { wv[q * (SCAN_STATIC_THREADS / 32) + w] = m; wi[q * (SCAN_STATIC_THREADS / 32) + w] = mi; }
    }
    if (lane == 0) wcnt[w] = nsw;
    __syncthreads();
    if (w == 0) {
        double v = wv[lane]; int bi = wi[lane];            // SCAN_STATIC_SPB / 32 == 32 slots
        warp_argmax_margin(v, bi);
        unsigned c = lane < SCAN_STATIC_THREADS / 32 ? wcnt[lane] : 0u;
        c = __reduce_add_sync(0xffffffffu, c);
        if (lane == 0) {
            cres[blockIdx.x].v = v; cres[blockIdx.x].idx = bi; cres[blockIdx.x].cnt = c;
            __threadfence();
            is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (!is_last) return;
    // the last CTA to finish reduces the per-CTA results (only the gridDim.x entries this launch wrote: whatever an
    // earlier, larger call left behind them is never read)
    __threadfence();
    double v = -CUDART_INF; int bi = 0x7fffffff;
    unsigned long long cnt = 0;
    for (int t = threadIdx.x; t < (int)gridDim.x; t += SCAN_STATIC_THREADS) {
        const double tv = __ldcg(&cres[t].v); const int ti = __ldcg(&cres[t].idx);
        cnt += __ldcg(&cres[t].cnt);
        if (better(tv, ti, v, bi)) { v = tv; bi = ti; }
    }
    warp_argmax_margin(v, bi);
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    __syncthreads();                                       // wv / wi are reused
    if (lane == 0) { wv[w] = v; wi[w] = bi; wc[w] = cnt; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < SCAN_STATIC_THREADS / 32; ++k) {
            if (better(wv[k], wi[k], v, bi)) { v = wv[k]; bi = wi[k]; }
            cnt += wc[k];
        }
        const bool any = v > 1.0;
        result[0] = (long long)cnt;
        result[1] = any ? bi : -1;
        reinterpret_cast<double*>(result)[2] = any ? v : -CUDART_INF;
        *ticket = 0u;                                      // leave the counter at zero (the entry point clears it as well)
    }
}

// Device address of g_scan_static_scratch on the CURRENT device: asked for once per device, with that device current,
// and kept.  cudaGetSymbolAddress loads this module on the device if nothing has yet (no cudaMalloc of ours).
std::mutex g_static_mutex;
unsigned char* g_static_scratch_dev[64] = {nullptr};
int static_scratch_of(int dev, unsigned char** out) {
    if (dev < 0 || dev >= 64) return fail(FS_ERR_CUDA, "device ordinal %d outside the table of 64", dev);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_scratch_dev[dev]) {
        void* p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&p, g_scan_static_scratch));
        if (!p) return fail(FS_ERR_CUDA, "cudaGetSymbolAddress returned a null address for the static scan scratch");
        g_static_scratch_dev[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_scratch_dev[dev];
    return FS_OK;
}

}  // namespace

extern "C" {

int fs_scan_static(int64_t N, const double* angle_dev, const double* hc_dev, const int8_t* s_dev, const double* hdip_dev,
                   const fs_params* p, double hx, double hy, double sigma_th, uint64_t seed, uint32_t step,
                   void* result_dev, void* stream) {
    if (N <= 0) return fail(FS_ERR_ARG, "N=%lld must be positive", (long long)N);
    if (N > (int64_t)FS_SCAN_STATIC_MAX_N)
        return fail(FS_ERR_ARG, "N=%lld exceeds FS_SCAN_STATIC_MAX_N=%d, the most the static scratch array holds "
                    "(use fs_create + fs_scan with a caller-allocated workspace for larger systems)", (long long)N,
                    (int)FS_SCAN_STATIC_MAX_N);
    if (!angle_dev || !hc_dev || !s_dev || !hdip_dev || !p || !result_dev) return fail(FS_ERR_ARG, "null pointer argument");
    if (!(p->b > 0) || !(p->c > 0) || !(p->beta > 0) || !(p->gamma > 0)) return fail(FS_ERR_ARG, "b, c, beta, gamma must be > 0");
    if (!(sigma_th >= 0) || !std::isfinite(sigma_th)) return fail(FS_ERR_ARG, "sigma_th must be finite and >= 0");
    if (((uintptr_t)result_dev & 7) || ((uintptr_t)hdip_dev & 15)) return fail(FS_ERR_ARG, "result_dev needs 8-byte, hdip_dev 16-byte alignment");
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    unsigned char* scratch = nullptr;
    int rc = static_scratch_of(dev, &scratch);
    if (rc) return rc;
    auto kind = [](double denom) { return denom == 3.0 ? 1 : (denom == 2.0 ? 2 : (denom == 1.0 ? 3 : 0)); };
    const Astroid ast{1.0 / p->b, 1.0 / p->c, 2.0 / p->gamma, 2.0 / p->beta, kind(p->gamma), kind(p->beta),
                      std::pow(0.5, p->gamma / 2.0) * (1.0 - 1e-9), std::pow(0.5, p->beta / 2.0) * (1.0 - 1e-9)};
    const FieldSpec fs{sigma_th, seed, step};
    cudaStream_t st = (cudaStream_t)stream;
    // the ticket counter must start at zero whatever an earlier (possibly failed) call left in the shared array
    CUDA_TRY(cudaMemsetAsync(scratch, 0, SCAN_STATIC_HEADER, st));
    const int ncta = (int)((N + SCAN_STATIC_SPB - 1) / SCAN_STATIC_SPB);
    k_scan_static<<<ncta, SCAN_STATIC_THREADS, 0, st>>>(N, ast, fs, make_double2(hx, hy), angle_dev, hc_dev, s_dev,
                                                        reinterpret_cast<const double2*>(hdip_dev), scratch,
                                                        static_cast<long long*>(result_dev));
    LAUNCHED();
    CUDA_TRY(cudaGetLastError());
    return FS_OK;
}

}  // extern "C"
