// field_fft.cu -- a1, spectral route ("more efficient
// parallelization of the dipole sum"): the dipole field as a batched circular convolution by FFT,
// organised around the checkerboard: every transform is a HALF-size transform of one colour.
//
//   h_n^a = sum_m W^{ab}(m - n) s_m^b  =>  h^(k) = M(k) s^(k),  M^{ab}(k) = sum_rho W^{ab}(rho) e^{+i k.rho}
//
// Colour c = (x + y) & 1 holds the sites x = 2 i + p_c(y), p_c(y) = (y + c) & 1, i in [0, L/2): the dense array
// S[c][a][y L/2 + i][r] of the internal layout.  Its transform
//   S^_c(kx, ky) = sum_y e^{-2 pi i ky y / L} e^{-2 pi i kx p_c(y) / L} G_{c,y}(kx),   G_{c,y} = (L/2)-point FFT of row y over i,
// obeys S^_c(kx + L/2, ky) = (-1)^c S^_c(kx, ky + L/2), so kx in [0, L/2) carries everything ("half-spectrum": N/2 values),
// and the field at the sites of colour t needs only the folded spectrum
//   H^_t(kx, ky) = h^(kx, ky) + (-1)^t h^(kx + L/2, ky + L/2) = A(kx, ky) S^_t(kx, ky) + B(kx, ky) S^_{1-t}(kx, ky),
//   A = M(k) + M(k + (L/2, L/2))  (displacements of even parity: same colour),  B = M(k) - M(k + (L/2, L/2))  (odd parity),
//   h_t(i, y) = (1/N) sum_{kx < L/2} e^{2 pi i kx i / (L/2)} e^{+2 pi i kx p_t(y) / L} sum_ky H^_t(kx, ky) e^{2 pi i ky y / L}.
// A checkerboard half-sweep of colour t changes only colour t, so in a running sweep the half-spectrum of the colour
// that was just updated is the only thing to recompute: S^_t from the half-sweep before last is still valid and is kept
// in a cache (C).  One field = three kernels, each a half-size pass:
//   fftc_x_forward   rows of the updated colour: (L/2)-point FFT over i, row phase, -> Z[a][slot_x][pb][y][lane]
//   fftc_y           columns kx < L/2: L-point FFT over y -> S^_{1-t} (stored to the cache), H^_t = A S^_t + B S^_{1-t},
//                    inverse L-point FFT over ky, in place in Z
//   fftc_x_inverse   rows of the target colour: row phase, inverse (L/2)-point FFT -> H (colour t only, dense)
// i.e. 2 half-size 2-D transforms per field where the full-lattice formulation needs 1 full forward + 1 full inverse.
//
// W is real, so the whole map s -> h is a real linear operator and two replicas ride through every complex transform as
// real and imaginary part: replicas r, r+1 are adjacent floats of the [c][a][site][r] layout, i.e. the spin array already
// IS an array of complex "replica pairs".  M may be complex (W need not be even).
// A length-n transform (n = 16 * N2) is the four-step algorithm: 16-point FFTs in registers over the stride-N2
// sub-sequences, twiddle, one pass through shared memory, N2-point FFTs in registers; spectra stay in "slot order"
// slot(k) = N2 (k mod 16) + k div 16 and the inverse runs the steps backwards, so no reordering pass exists anywhere and
// A, B are tabulated in slot order with the 1/N of the inverse folded in.
#include "metropolis_pair.cuh"
#include "bulk_copy.cuh"

namespace {

// ---- compile-time twiddles ------------------------------------------------------------------
constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double c_sin_small(double x) {  // |x| <= pi/4
    double term = x, sum = x;
    for (int i = 1; i < 14; ++i) {
        term *= -x * x / ((2.0 * i) * (2.0 * i + 1.0));
        sum += term;
    }
    return sum;
}
constexpr double c_cos_small(double x) {
    double term = 1.0, sum = 1.0;
    for (int i = 1; i < 14; ++i) {
        term *= -x * x / ((2.0 * i - 1.0) * (2.0 * i));
        sum += term;
    }
    return sum;
}
// cos and sin of 2 pi k / n for 0 <= k < n, n a power of two >= 8, by octant reduction
constexpr double c_cos2pi(int k, int n) {
    k %= n;
    if (k > n / 2) k = n - k;                       // cos is even about pi
    if (k > n / 4) return -c_cos2pi(n / 2 - k, n);  // cos(pi - x) = -cos x
    if (k > n / 8) return c_sin_small(2.0 * kPi * (n / 4 - k) / n);
    return c_cos_small(2.0 * kPi * k / n);
}
constexpr double c_sin2pi(int k, int n) { return c_cos2pi(k + 3 * (n / 4), n); }  // sin x = cos(x - pi/2)

struct TwTable {
    float c[32], s[32];
};
constexpr TwTable make_tw32() {
    TwTable t{};
    for (int k = 0; k < 32; ++k) {
        t.c[k] = (float)c_cos2pi(k, 32);
        t.s[k] = (float)c_sin2pi(k, 32);
    }
    return t;
}
__device__ constexpr TwTable kTw32 = make_tw32();

// complex add / subtract as one packed instruction (FADD2 / FFMA2 with -1): the same IEEE results as two scalar
// adds, half the issue slots (fft field 71.8 -> 69.0 us at L = 256, R = 64; packing the twiddle multiplies as
// FMUL2 + FFMA2 as well was measured slower, 75.1 us, and is not done)
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2, %3}; mov.b64 rb, {%4, %5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0, %1}, rc; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc, rm; mov.b64 ra, {%2, %3}; mov.b64 rb, {%4, %5}; mov.b64 rm, {%6, %6}; fma.rn.f32x2 rc, rb, rm, ra; mov.b64 {%0, %1}, rc; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(-1.0f));
    return r;
}
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
}

template <int N>
__host__ __device__ constexpr int bitrev(int k) {
    int r = 0;
    for (int b = 1; b < N; b <<= 1) {
        r = (r << 1) | (k & 1);
        k >>= 1;
    }
    return r;
}

// In-register radix-2 decimation-in-frequency FFT of N <= 32 points; forward = e^{-2 pi i jk/N},
// INV conjugates the twiddles (no scaling).  Output: v[bitrev(k)] = X[k].  Everything unrolls;
// the twiddle of a butterfly is a compile-time constant and the trivial ones (1, -i) cost nothing.
template <int N, bool INV>
__device__ __forceinline__ void fft_reg(float2 (&v)[N]) {
#pragma unroll
    for (int len = N; len >= 2; len >>= 1) {
        const int half = len >> 1;
#pragma unroll
        for (int base = 0; base < N; base += len) {
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const float2 a = v[base + j], b = v[base + j + half];
                v[base + j] = cadd(a, b);
                const float2 d = csub(a, b);
                if (j == 0) {
                    v[base + j + half] = d;
                } else if (4 * j == len) {            // w = -i (forward), +i (inverse)
                    v[base + j + half] = INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
                } else {
                    const int t = j * (32 / len);     // index into the 32-point table
                    const float wc = kTw32.c[t], ws = INV ? kTw32.s[t] : -kTw32.s[t];
                    v[base + j + half] = cmul(d, make_float2(wc, ws));
                }
            }
        }
    }
}

// ---- the four steps of a length n = 16 * N2 transform --------------------------------------
// Twiddles come from two tables of L entries (L = the LATTICE size; a length-L line uses stride TS = 1, a length-L/2 line
// TS = 2): twf[j] = (c, -s) = e^{-2 pi i j / L} (forward transforms), twi[j] = (c, s) (inverse transforms), read with
// 64-bit shared loads (128-bit entries holding both operand pairs of the packed multiply were measured slower: a
// broadcast LDS.128 still takes four passes, and the x passes became bound by the shared-memory queue).
// a * (x + i y) = a.x (x, y) + a.y (-y, x): one sign flip (integer pipe), one FMUL2 and one FFMA2 with the scalars as
// broadcast operands.
__device__ __forceinline__ float2 cmul_tw(float2 a, float2 w) {
    f2 r = f2_mul(f2_bc(a.x), f2_make(w.x, w.y));
    r = f2_fma(f2_bc(a.y), f2_make(__uint_as_float(__float_as_uint(w.y) ^ 0x80000000u), w.x), r);
    float2 o;
    f2_split(r, o.x, o.y);
    return o;
}

// LNC = lanes (replica pairs) per line as a compile-time constant, 0 = blockDim.x (small replica counts)
template <int LNC>
__device__ __forceinline__ int nlanes() { return LNC ? LNC : (int)blockDim.x; }

// x passes: buf[sidx(k1, n2) * LN + lane] is the CTA's shared line buffer: slot N2 k1 + n2 with one pad row per block of
// N2 slots, so that blocks k1, k1 + 1 of a warp fall on different banks when LN < 16.  Threads are (lane, t).
template <int N2>
__device__ __forceinline__ int sidx(int k1, int n2) { return (N2 + 1) * k1 + n2; }
template <int N2>
__host__ __device__ constexpr int line_rows() { return (N2 + 1) * 16; }

// forward step 1: v[n1] = x[N2 n1 + n2]  ->  A[k1][n2] * W_n^{n2 k1}  at slot N2 k1 + n2
template <int N2, int TS, int LNC>
__device__ __forceinline__ void fwd_step1(float2 (&v)[16], int n2, const float2 *twf, float2 *buf, int lane) {
    const int LN = nlanes<LNC>();
    float2 w[16];                                          // all twiddles first: the loads go out as one batch
#pragma unroll
    for (int k1 = 1; k1 < 16; ++k1) w[k1] = twf[TS * n2 * k1];
    fft_reg<16, false>(v);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1)
        buf[sidx<N2>(k1, n2) * LN + lane] = k1 == 0 ? v[0] : cmul_tw(v[bitrev<16>(k1)], w[k1]);
}
// forward step 2: block k1 -> u[k2] = X[k1 + 16 k2] in natural k2 order
template <int N2, int LNC>
__device__ __forceinline__ void fwd_step2(float2 (&u)[N2], int k1, const float2 *buf, int lane) {
    const int LN = nlanes<LNC>();
    float2 t[N2];
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2) t[n2] = buf[sidx<N2>(k1, n2) * LN + lane];
    fft_reg<N2, false>(t);
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) u[k2] = t[bitrev<N2>(k2)];
}
// inverse step 2: u[k2] = Y[k1 + 16 k2]  ->  B[k1][n2] * conj(W_n^{n2 k1})  at slot N2 k1 + n2
template <int N2, int TS, int LNC>
__device__ __forceinline__ void inv_step2(float2 (&u)[N2], int k1, const float2 *twi, float2 *buf, int lane) {
    const int LN = nlanes<LNC>();
    float2 w[N2];
#pragma unroll
    for (int n2 = 1; n2 < N2; ++n2) w[n2] = twi[TS * n2 * k1];
    fft_reg<N2, true>(u);
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2)
        buf[sidx<N2>(k1, n2) * LN + lane] = n2 == 0 ? u[0] : cmul_tw(u[bitrev<N2>(n2)], w[n2]);
}
// inverse step 1: slots N2 k1 + n2 (k1 = 0..15)  ->  v[n1] = x[N2 n1 + n2]
template <int N2, int LNC>
__device__ __forceinline__ void inv_step1(float2 (&v)[16], int n2, const float2 *buf, int lane) {
    const int LN = nlanes<LNC>();
    float2 t[16];
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) t[k1] = buf[sidx<N2>(k1, n2) * LN + lane];
    fft_reg<16, true>(t);
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) v[n1] = t[bitrev<16>(n1)];
}

// Z and the two caches share one layout: [a][slot_x][pb][row'][lane], a = component, slot_x < L/2, pb = block of LZ
// replica pairs (LZ <= 8), row = y (Z after the x pass / before the x-inverse pass) or slot_y (spectra), lane = pair
// within the block.  One (a, slot_x, pb) line is L * LZ contiguous complex numbers: one TMA bulk copy moves it between
// global and shared memory, where the y pass transforms it in place.  row' = row ^ ((row >> 4) & 1): with 8-byte
// elements and LZ = 8 a row is 64 bytes = 16 banks, rows of equal parity share banks, and the second step of the
// four-step transform has the threads of a half-warp read rows 16 apart; the swap of neighbouring rows in every other
// block of 16 puts them on different banks (the first step reads runs of consecutive rows either way).
struct FcParams {
    const float *S;    // spins, internal layout
    float *H;          // field, internal layout
    float2 *Z;         // scratch lines of the field being computed
    float2 *Cnew;      // y pass: cache of the half-spectrum of colour `colour` (written unless FC_COMBINE, then read)
    const float2 *Ctgt;  // y pass: cache of the half-spectrum of the target colour 1 - colour
    const float4 *AB;  // AB[slot_x][slot_y][4]: (Axx, Axy), (Ayy, Bxx), (Bxy, Byy), (Azz, Bzz), each complex, scaled 1/N
    const float2 *twf, *twi;  // twiddle tables, L entries each (behind AB in the workspace)
    int L, P;          // P = R / 2 complex replica pairs
    int LZ, PBZ;       // lanes per line and line blocks: P = PBZ * LZ
    int pb0;           // y pass and fused row kernel: first line block of this launch (grid.x = line blocks it covers)
    float *SG;         // fused row kernel: null, or the block-major copy of the spins SG[pb][q][c][a][lane] to work on
    int colour;        // x passes: the colour of the rows; y pass: the colour whose lines sit in Z / in Cnew
};

__device__ __forceinline__ int swz(int row) { return row ^ ((row >> 4) & 1); }
__device__ __forceinline__ size_t line_base(const FcParams &p, int a, int sx, int pb) {
    return ((((size_t)a * (p.L >> 1) + sx) * p.PBZ + pb) * p.L) * p.LZ;
}

// x forward, colour p.colour: grid (P / LN, L rows, 3 components), block (LN, TL), TL = min(16, N2X) threads per line.
template <int N2X, int LNC>
__global__ void __launch_bounds__(256) fftc_x_forward_kernel(const FcParams p) {
    extern __shared__ __align__(16) float2 fsm[];
    constexpr int Lh = 16 * N2X, L = 2 * Lh;
    const int LN = nlanes<LNC>(), TL = blockDim.y;
    float2 *twf = fsm, *buf = fsm + L;
    const int lane = threadIdx.x, t = threadIdx.y, tid = t * LN + lane;
    const int pair = blockIdx.x * LN + lane, y = blockIdx.y, a = blockIdx.z, c = p.colour;
    for (int j = tid; j < L; j += LN * TL) twf[j] = __ldg(p.twf + j);   // a constant table: before the wait
    const size_t planeP = (size_t)L * Lh * p.P;
    const float2 *src = reinterpret_cast<const float2 *>(p.S) + (size_t)(c * 3 + a) * planeP + (size_t)y * Lh * p.P + pair;
    const unsigned ld_stride = (unsigned)(N2X * p.P);
    pdl_wait();                                            // the spins come from the Metropolis kernel before
    float2 v[16];
    src += (unsigned)t * p.P;                              // t < N2X by construction
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) v[n1] = __ldg(src + n1 * ld_stride);
    __syncthreads();
    fwd_step1<N2X, 2, LNC>(v, t, twf, buf, lane);
    __syncthreads();
    pdl_trigger();                                         // late: a successor resident earlier only takes room
    const bool odd_row = (y + c) & 1;                      // sites x = 2 i + 1: row phase e^{-2 pi i kx / L}
    const int lz = LNC ? (LNC < 8 ? LNC : 8) : p.LZ;       // LNC = 16 goes with lines of 8 pairs
    float2 *dst = p.Z + line_base(p, a, 0, pair / lz) + (size_t)swz(y) * lz + pair % lz;
    const unsigned sx_stride = (unsigned)(p.PBZ * L * lz);
    for (int k1 = t; k1 < 16; k1 += TL) {
        float2 u[N2X], w[N2X];
#pragma unroll
        for (int k2 = 0; k2 < N2X; ++k2) w[k2] = twf[odd_row ? k1 + 16 * k2 : 0];   // twf[0] = 1: no branch
        fwd_step2<N2X, LNC>(u, k1, buf, lane);
#pragma unroll
        for (int k2 = 0; k2 < N2X; ++k2) dst[(unsigned)(N2X * k1 + k2) * sx_stride] = cmul_tw(u[k2], w[k2]);
    }
}

// x inverse, target colour p.colour: grid (P / LN, L rows, 3 components), block (LN, TL).
template <int N2X, int LNC>
__global__ void __launch_bounds__(256) fftc_x_inverse_kernel(const FcParams p) {
    extern __shared__ __align__(16) float2 fsm[];
    constexpr int Lh = 16 * N2X, L = 2 * Lh;
    const int LN = nlanes<LNC>(), TL = blockDim.y;
    float2 *twi = fsm, *buf = fsm + L;
    const int lane = threadIdx.x, t = threadIdx.y, tid = t * LN + lane;
    const int pair = blockIdx.x * LN + lane, y = blockIdx.y, a = blockIdx.z, c = p.colour;
    for (int j = tid; j < L; j += LN * TL) twi[j] = __ldg(p.twi + j);
    const int lz = LNC ? (LNC < 8 ? LNC : 8) : p.LZ;
    const float2 *src = p.Z + line_base(p, a, 0, pair / lz) + (size_t)swz(y) * lz + pair % lz;
    const unsigned sx_stride = (unsigned)(p.PBZ * L * lz);
    constexpr int NK = N2X >= 16 ? 1 : 16 / N2X;           // blocks k1 per thread
    pdl_wait();                                            // the lines come from the y pass
    float2 u[NK][N2X];
#pragma unroll
    for (int j = 0; j < NK; ++j)
#pragma unroll
        for (int k2 = 0; k2 < N2X; ++k2) u[j][k2] = src[(unsigned)(N2X * (t + j * TL) + k2) * sx_stride];
    __syncthreads();
    const bool odd_row = (y + c) & 1;                      // row phase e^{+2 pi i kx / L}
#pragma unroll
    for (int j = 0; j < NK; ++j) {
        const int k1 = t + j * TL;
        float2 w[N2X];
#pragma unroll
        for (int k2 = 0; k2 < N2X; ++k2) w[k2] = twi[odd_row ? k1 + 16 * k2 : 0];   // twi[0] = 1: no branch
#pragma unroll
        for (int k2 = 0; k2 < N2X; ++k2) u[j][k2] = cmul_tw(u[j][k2], w[k2]);
        inv_step2<N2X, 2, LNC>(u[j], k1, twi, buf, lane);
    }
    pdl_trigger();
    __syncthreads();
    float2 v[16];
    inv_step1<N2X, LNC>(v, t, buf, lane);
    const size_t planeP = (size_t)L * Lh * p.P;
    float2 *dst = reinterpret_cast<float2 *>(p.H) + (size_t)(c * 3 + a) * planeP + (size_t)y * Lh * p.P + pair + (unsigned)t * p.P;
    const unsigned st_stride = (unsigned)(N2X * p.P);
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) dst[n1 * st_stride] = v[n1];
}

// The fused row kernel of a running FFT sweep: everything a half-sweep of colour t does to one lattice row, in one launch.
//   A. x inverse of the three components (as fftc_x_inverse_kernel), the field h of the row left in shared memory;
//   B. the Metropolis decision of every site of the row (metropolis_pair.cuh: the arithmetic of metropolis4_kernel, pair by
//      pair, on the same inputs in the same order -- bit-identical decisions), new spins to the spin array and to shared
//      memory;
//   C. x forward of the UPDATED row (as fftc_x_forward_kernel), written over the row's entries of Z: the lines the next
//      field's y pass needs (colour t is then the colour that was just updated).
// A half-sweep is then two launches (y pass, this kernel) instead of four, h is never written to or read from global
// memory, and the updated spins are transformed while they are on the chip.
//   grid (P / LN, L rows), block (LN, TL, 3 components); LN = the line width LZ (8 at config 5).
// Phase B's items (site i, pair) are spread over all threads; every other phase works on component threadIdx.z.
template <int N2X, int LNC, bool DEVSTEP, int FLIP>
__global__ void __launch_bounds__(N2X >= 16 ? 384 : 192, N2X >= 16 ? 2 : 4) fftc_row_update_kernel(const FcParams p, const MetropolisArgs ma, const RoundKeys rk) {
    extern __shared__ __align__(16) float2 fsm[];
    constexpr int Lh = 16 * N2X, L = 2 * Lh;
    const int LN = nlanes<LNC>(), TL = blockDim.y;
    float2 *twi = fsm, *twf = fsm + L;
    const int lane = threadIdx.x, t = threadIdx.y, a = threadIdx.z;
    const int nthr = LN * TL * 3, tid = (a * TL + t) * LN + lane;
    float2 *X0 = fsm + 2 * L;                              // three exchange buffers, also h / spins of the row by site
    const int xstride = line_rows<N2X>() * LN;
    float2 *buf = X0 + a * xstride;
    const int pb = blockIdx.x + p.pb0, y = blockIdx.y, c = p.colour;
    for (int j = tid; j < L; j += nthr) twi[j] = __ldg(p.twi + j), twf[j] = __ldg(p.twf + j);   // constant tables
    float2 *zline = p.Z + line_base(p, a, 0, pb) + (size_t)swz(y) * LN + lane;   // LN == p.LZ
    const unsigned sx_stride = (unsigned)(p.PBZ * L * LN);
    constexpr int NK = N2X >= 16 ? 1 : 16 / N2X;           // blocks k1 per thread
    const bool odd_row = (y + c) & 1;
    pdl_wait();                                            // the lines come from the y pass, the spins from earlier kernels
    // ---- A: x inverse -> h(i) of this component in buf[i * LN + lane]
    {
        float2 u[NK][N2X];
#pragma unroll
        for (int j = 0; j < NK; ++j)
#pragma unroll
            for (int k2 = 0; k2 < N2X; ++k2) u[j][k2] = zline[(unsigned)(N2X * (t + j * TL) + k2) * sx_stride];
        __syncthreads();
#pragma unroll
        for (int j = 0; j < NK; ++j) {
            const int k1 = t + j * TL;
            float2 w[N2X];
#pragma unroll
            for (int k2 = 0; k2 < N2X; ++k2) w[k2] = twi[odd_row ? k1 + 16 * k2 : 0];
#pragma unroll
            for (int k2 = 0; k2 < N2X; ++k2) u[j][k2] = cmul_tw(u[j][k2], w[k2]);
            inv_step2<N2X, 2, LNC>(u[j], k1, twi, buf, lane);
        }
        __syncthreads();
        float2 v[16];
        inv_step1<N2X, LNC>(v, t, buf, lane);
        __syncthreads();                                   // everybody has read the exchange layout: reuse it by site
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) buf[(N2X * n1 + t) * LN + lane] = v[n1];
    }
    __syncthreads();
    // ---- B: Metropolis on the row (eq. 7; the half-sweep's frozen field is the h just computed)
    {
        // the spins: the internal array (replica pairs of all line blocks side by side: runs of LN pairs = 64 bytes, P pairs
        // apart) or, for a chain of the branched replay, the chain's line block in the block-major copy SG (dense)
        const bool dense = p.SG != nullptr;
        const int Pe = dense ? LN : p.P;
        const int pr_sub = dense ? pb * LN : 0;               // pair index within the spin record: pr, or the lane in the block's copy
        const size_t planeP = (size_t)L * Lh * Pe;
        f2 *S2 = dense ? reinterpret_cast<f2 *>(p.SG) + (size_t)pb * 6 * planeP : reinterpret_cast<f2 *>(ma.S);
        const f2 *X2 = reinterpret_cast<const f2 *>(X0);
        f2 *X2w = reinterpret_cast<f2 *>(X0);
        const int yn = (y + 1 == L) ? 0 : y + 1, ys = (y == 0) ? L - 1 : y - 1;
        const size_t own0 = (size_t)c * 3 * planeP + (size_t)y * Lh * Pe, oth = (size_t)(1 - c) * 3 * planeP;
        const size_t o0 = oth + (size_t)y * Lh * Pe, on = oth + (size_t)yn * Lh * Pe, os = oth + (size_t)ys * Lh * Pe;
        uint32_t step_lo = ma.step_lo, step_hi = ma.step_hi;
        if (DEVSTEP) step_words(ma, step_lo, step_hi);
        for (int item = tid; item < Lh * LN; item += nthr) {
            const int i = item / LN, ln = item - i * LN, pr = pb * LN + ln;
            const int i1 = odd_row ? (i + 1 == Lh ? 0 : i + 1) : (i == 0 ? Lh - 1 : i - 1);
            const unsigned e = (unsigned)(i * Pe + pr - pr_sub), e1 = (unsigned)(i1 * Pe + pr - pr_sub);
            f2 s[3], nb[3], h[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                s[k] = S2[own0 + k * planeP + e];
                const f2 va = __ldg(S2 + o0 + k * planeP + e), vb = __ldg(S2 + o0 + k * planeP + e1);
                const f2 vc = __ldg(S2 + on + k * planeP + e), vd = __ldg(S2 + os + k * planeP + e);
                nb[k] = f2_add(f2_add(va, vb), f2_add(vc, vd));
                h[k] = X2[k * xstride + item];
            }
            const f2 invT = __ldg(reinterpret_cast<const f2 *>(ma.invT) + pr), K2 = __ldg(reinterpret_cast<const f2 *>(ma.K2) + pr),
                     K4 = __ldg(reinterpret_cast<const f2 *>(ma.K4) + pr);
            const uint32_t n = (uint32_t)(y * L + 2 * i + (odd_row ? 1 : 0));
            const uint32_t r = 2u * (uint32_t)pr + ma.r_off;
            const uint4 ra = philox4x32_10(make_uint4(n, r, step_lo, step_hi), rk);
            const uint4 rb = philox4x32_10(make_uint4(n, r + 1u, step_lo, step_hi), rk);
            Trial2 tr = trial2(ra, rb);
            if (FLIP) {                                    // Ising move of App. B: complete reversal
                tr.tx = f2_mul(s[0], f2_bc(-1.0f));
                tr.ty = f2_mul(s[1], f2_bc(-1.0f));
                tr.tz = f2_mul(s[2], f2_bc(-1.0f));
            }
            const f2 margin = margin2(ma, tr, s[0], s[1], s[2], nb[0], nb[1], nb[2], h[0], h[1], h[2], invT, K2, K4);
            float m0, m1;
            f2_split(margin, m0, m1);
            const bool acc0 = m0 < 0.0f, acc1 = m1 < 0.0f;
            const f2 tv[3] = {tr.tx, tr.ty, tr.tz};
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                float a0, a1, b0, b1;
                f2_split(tv[k], a0, a1);
                f2_split(s[k], b0, b1);
                s[k] = f2_make(acc0 ? a0 : b0, acc1 ? a1 : b1);
                X2w[k * xstride + item] = s[k];            // the row after the update, for phase C
            }
            if (acc0 | acc1) {
#pragma unroll
                for (int k = 0; k < 3; ++k) S2[own0 + k * planeP + e] = s[k];
            }
        }
    }
    __syncthreads();
    // ---- C: x forward of the updated row -> the row's entries of Z
    {
        float2 v[16];
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) v[n1] = buf[(N2X * n1 + t) * LN + lane];
        __syncthreads();
        fwd_step1<N2X, 2, LNC>(v, t, twf, buf, lane);
        __syncthreads();
        pdl_trigger();
        for (int k1 = t; k1 < 16; k1 += TL) {
            float2 u[N2X], w[N2X];
#pragma unroll
            for (int k2 = 0; k2 < N2X; ++k2) w[k2] = twf[odd_row ? k1 + 16 * k2 : 0];
            fwd_step2<N2X, LNC>(u, k1, buf, lane);
#pragma unroll
            for (int k2 = 0; k2 < N2X; ++k2) zline[(unsigned)(N2X * k1 + k2) * sx_stride] = cmul_tw(u[k2], w[k2]);
        }
    }
}

// In-place four-step transforms of one shared-memory line B[row' * LZ + lane] (rows = y or slot_y, see FcParams).
// Forward: natural order in, slot order out; inverse: slot order in, natural order out.  Step 1 works on the rows
// {N2 n1 + n2 : n1} = {N2 k1 + n2 : k1} of a sub-sequence n2, step 2 on the rows {N2 t + k} of block t: both write back
// exactly the rows they read, so each half needs no barrier of its own (the caller puts one between the halves).
template <int N2, int LZC>
__device__ __forceinline__ void line_fwd_step1(float2 *B, const float2 *twf, int lane, int t) {
    const int LZ = nlanes<LZC>();
    for (int n2 = t; n2 < N2; n2 += 16) {
        float2 v[16], w[16];
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) v[n1] = B[swz(N2 * n1 + n2) * LZ + lane];
#pragma unroll
        for (int k1 = 1; k1 < 16; ++k1) w[k1] = twf[n2 * k1];
        fft_reg<16, false>(v);
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1)
            B[swz(N2 * k1 + n2) * LZ + lane] = k1 == 0 ? v[0] : cmul_tw(v[bitrev<16>(k1)], w[k1]);
    }
}
template <int N2, int LZC>
__device__ __forceinline__ void line_fwd_step2(float2 *B, int lane, int t) {
    const int LZ = nlanes<LZC>();
    float2 v[N2];
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2) v[n2] = B[swz(N2 * t + n2) * LZ + lane];
    fft_reg<N2, false>(v);
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) B[swz(N2 * t + k2) * LZ + lane] = v[bitrev<N2>(k2)];
}
template <int N2, int LZC>
__device__ __forceinline__ void line_inv_step2(float2 *B, const float2 *twi, int lane, int t) {
    const int LZ = nlanes<LZC>();
    float2 u[N2], w[N2];
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) u[k2] = B[swz(N2 * t + k2) * LZ + lane];
#pragma unroll
    for (int n2 = 1; n2 < N2; ++n2) w[n2] = twi[n2 * t];
    fft_reg<N2, true>(u);
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2)
        B[swz(N2 * t + n2) * LZ + lane] = n2 == 0 ? u[0] : cmul_tw(u[bitrev<N2>(n2)], w[n2]);
}
template <int N2, int LZC>
__device__ __forceinline__ void line_inv_step1(float2 *B, int lane, int t) {
    const int LZ = nlanes<LZC>();
    for (int n2 = t; n2 < N2; n2 += 16) {
        float2 v[16];
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) v[k1] = B[swz(N2 * k1 + n2) * LZ + lane];
        fft_reg<16, true>(v);
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) B[swz(N2 * n1 + n2) * LZ + lane] = v[bitrev<16>(n1)];
    }
}

// packed complex arithmetic of the spectral multiply: (a.x, a.y) as one 64-bit operand, m * a = m.x (a.x, a.y) + m.y (-a.y, a.x)
__device__ __forceinline__ f2 c_pack(float2 a) { return f2_make(a.x, a.y); }
__device__ __forceinline__ f2 c_rot(float2 a) { return f2_make(-a.y, a.x); }     // i * a
__device__ __forceinline__ f2 c_mac(f2 acc, float mre, float mim, f2 a, f2 ia) {  // acc + m * a
    return f2_fma(f2_bc(mim), ia, f2_fma(f2_bc(mre), a, acc));
}
__device__ __forceinline__ f2 c_mul(float mre, float mim, f2 a, f2 ia) { return f2_fma(f2_bc(mim), ia, f2_mul(f2_bc(mre), a)); }
__device__ __forceinline__ float2 c_unpack(f2 v) {
    float2 o;
    f2_split(v, o.x, o.y);
    return o;
}

// The y pass.  A CTA owns two lines of LZ replica pairs, one per half of its threads, and transforms them in place in
// shared memory; every byte it moves to or from global memory goes by TMA bulk copy (one contiguous line each, the
// twiddle tables too), issued by one thread at the top, so no warp ever waits on a global load except for the few
// table values of the spectral multiply.
//   grid (PBZ, L/2 + L/4), block (LZ, 16, 2).  blockIdx.y < L/2: the x and y lines of column slot_x = blockIdx.y (they mix
//   through W^xy); else the z lines of the two columns 2 (blockIdx.y - L/2) and + 1: every CTA has the same size.
//   FC_FWD_ONLY  Z holds the x-transformed rows of colour c = p.colour: forward L-point FFT over y -> S^_c -> Cnew.
//   FC_FUSED     the same, then H^_t = A S^_t + B S^_c with t = 1 - c and S^_t read from Ctgt, inverse FFT over ky -> Z.
//   FC_COMBINE   nothing to transform forward: S^_c is read from Cnew as well (both caches valid); t = 1 - c.
// The three modes run the same arithmetic on the same values, so a field does not depend on which of them produced it.
enum { FC_FWD_ONLY = 0, FC_FUSED = 1, FC_COMBINE = 2 };

template <int N2, int MODE, int LZC>
__global__ void __launch_bounds__(256, 3) fftc_y_kernel(const FcParams p) {
    extern __shared__ __align__(128) unsigned char ysm_raw[];
    constexpr int L = 16 * N2, Lh = L / 2;
    const int LZ = nlanes<LZC>();
    const uint32_t line_elems = (uint32_t)(L * LZ), line_bytes = line_elems * (uint32_t)sizeof(float2);
    constexpr uint32_t tw_bytes = (uint32_t)(L * sizeof(float2));
    float2 *B0 = reinterpret_cast<float2 *>(ysm_raw), *B1 = B0 + line_elems, *B2 = B1 + line_elems, *B3 = B2 + line_elems;
    float2 *twf = B0 + (MODE == FC_FWD_ONLY ? 2 : 4) * (size_t)line_elems, *twi = twf + L;
    uint64_t *bars = reinterpret_cast<uint64_t *>(twi + L);
    const int lane = threadIdx.x, t = threadIdx.y, j = threadIdx.z, tid = (j * 16 + t) * LZ + lane;
    const int pb = blockIdx.x + p.pb0;
    const bool is_z = (int)blockIdx.y >= Lh;
    const int sx0 = is_z ? 2 * ((int)blockIdx.y - Lh) : (int)blockIdx.y;
    const int sx1 = is_z ? sx0 + 1 : sx0;
    const size_t off0 = line_base(p, is_z ? 2 : 0, sx0, pb), off1 = line_base(p, is_z ? 2 : 1, sx1, pb);
    if (tid == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_wait();                                            // Z comes from the x pass, the caches from earlier y passes
    if (tid == 0) {
        const float2 *in = MODE == FC_COMBINE ? p.Cnew : p.Z;
        mbar_expect_tx(&bars[0], 2 * line_bytes + (MODE == FC_COMBINE ? 0 : tw_bytes));
        if (MODE != FC_COMBINE) bulk_g2s(twf, p.twf, tw_bytes, &bars[0]);
        bulk_g2s(B0, in + off0, line_bytes, &bars[0]);
        bulk_g2s(B1, in + off1, line_bytes, &bars[0]);
        if (MODE != FC_FWD_ONLY) {
            mbar_expect_tx(&bars[1], 2 * line_bytes + tw_bytes);
            bulk_g2s(twi, p.twi, tw_bytes, &bars[1]);
            // The cached spectra stream through the L2 (evict_first on their loads and stores): a cache line of S^_t is read
            // exactly once, a half-sweep after it was written, and rewritten a half-sweep later.  At config 5 the spins
            // (50 MB), Z (25 MB) and the two caches (50 MB) together are the size of the L2; without the hint the
            // cyclic access pattern evicts all of it in turn, with it the spins and Z stay resident (measured: 89.5 ->
            // 84.7 us per sweep; hints on the Z lines or evict_last on anything gained nothing).
            const uint64_t stream_pol = l2_policy_evict_first();
            bulk_g2s_hint(B2, p.Ctgt + off0, line_bytes, &bars[1], stream_pol);
            bulk_g2s_hint(B3, p.Ctgt + off1, line_bytes, &bars[1], stream_pol);
        }
    }
    mbar_wait(&bars[0], 0);
    if (MODE != FC_COMBINE) {
        float2 *Bj = j ? B1 : B0;                          // the two lines side by side, one per half of the threads
        line_fwd_step1<N2, LZC>(Bj, twf, lane, t);
        __syncthreads();
        line_fwd_step2<N2, LZC>(Bj, lane, t);
        fence_async_smem();                                // the spectra go to the cache straight from shared memory
        __syncthreads();
        if (tid == 0) {
            const uint64_t stream_pol = l2_policy_evict_first();
            bulk_s2g_hint(p.Cnew + off0, B0, line_bytes, stream_pol);
            bulk_s2g_hint(p.Cnew + off1, B1, line_bytes, stream_pol);
            bulk_commit();
        }
        if (MODE == FC_FWD_ONLY) {
            pdl_trigger();
            if (tid == 0) bulk_wait_all();
            return;
        }
    }
    mbar_wait(&bars[1], 0);
    // H^ = A S^_t + B S^_c on the rows N2 t + k2 (half of the k2 for each half of the threads), result over S^_t in B2, B3
    constexpr int KH = N2 / 2;
    if (!is_z) {
        const float4 *tab = p.AB + ((size_t)sx0 * L + N2 * t + KH * j) * 4;   // constant table, read-only path
#pragma unroll 4
        for (int k2 = 0; k2 < KH; ++k2) {
            const float4 m0 = __ldg(tab + 4 * k2), m1 = __ldg(tab + 4 * k2 + 1), m2 = __ldg(tab + 4 * k2 + 2);
            const int r = swz(N2 * t + KH * j + k2) * LZ + lane;
            const float2 ox = B0[r], oy = B1[r], tx = B2[r], ty = B3[r];
            const f2 pox = c_pack(ox), poy = c_pack(oy), ptx = c_pack(tx), pty = c_pack(ty);
            const f2 iox = c_rot(ox), ioy = c_rot(oy), itx = c_rot(tx), ity = c_rot(ty);
            // (Axx, Axy) = m0, (Ayy, Bxx) = m1, (Bxy, Byy) = m2
            f2 hx = c_mul(m0.x, m0.y, ptx, itx);
            hx = c_mac(hx, m0.z, m0.w, pty, ity);
            hx = c_mac(hx, m1.z, m1.w, pox, iox);
            hx = c_mac(hx, m2.x, m2.y, poy, ioy);
            f2 hy = c_mul(m0.z, m0.w, ptx, itx);
            hy = c_mac(hy, m1.x, m1.y, pty, ity);
            hy = c_mac(hy, m2.x, m2.y, pox, iox);
            hy = c_mac(hy, m2.z, m2.w, poy, ioy);
            B2[r] = c_unpack(hx);
            B3[r] = c_unpack(hy);
        }
    } else {
        const float4 *tab0 = p.AB + ((size_t)sx0 * L + N2 * t + KH * j) * 4 + 3;
        const float4 *tab1 = p.AB + ((size_t)sx1 * L + N2 * t + KH * j) * 4 + 3;
#pragma unroll 4
        for (int k2 = 0; k2 < KH; ++k2) {
            const float4 ma = __ldg(tab0 + 4 * k2), mb = __ldg(tab1 + 4 * k2);   // (Azz, Bzz) of the two columns
            const int r = swz(N2 * t + KH * j + k2) * LZ + lane;
            const float2 o0 = B0[r], o1 = B1[r], t0 = B2[r], t1 = B3[r];
            B2[r] = c_unpack(c_mac(c_mul(ma.x, ma.y, c_pack(t0), c_rot(t0)), ma.z, ma.w, c_pack(o0), c_rot(o0)));
            B3[r] = c_unpack(c_mac(c_mul(mb.x, mb.y, c_pack(t1), c_rot(t1)), mb.z, mb.w, c_pack(o1), c_rot(o1)));
        }
    }
    __syncthreads();
    float2 *Bj = j ? B3 : B2;
    line_inv_step2<N2, LZC>(Bj, twi, lane, t);
    __syncthreads();
    line_inv_step1<N2, LZC>(Bj, lane, t);
    fence_async_smem();
    __syncthreads();
    pdl_trigger();
    if (tid == 0) {
        bulk_s2g(p.Z + off0, B2, line_bytes);
        bulk_s2g(p.Z + off1, B3, line_bytes);
        bulk_commit();
        bulk_wait_all();                                   // shared memory must outlive the copies; the next kernel reads Z
    }
}

// ---- A, B = folded transform of W, fp64, once per tensor --------------------------------------
// T1[c][rho_y][kx] = sum_{rho_x} W[c][rho_y][rho_x] e^{+2 pi i kx rho_x / L}
__global__ void wq_pass1_kernel(const float *__restrict__ Wc, double2 *__restrict__ T1, int L) {
    const size_t N = (size_t)L * L;
    const size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= 4 * N) return;
    const int kx = (int)(id % L);
    const float *row = Wc + (id / L) * L;              // (c, rho_y) row
    double re = 0.0, im = 0.0;
    for (int rx = 0; rx < L; ++rx) {
        double s, c;
        sincospi(2.0 * (double)((kx * rx) % L) / (double)L, &s, &c);
        const double w = (double)row[rx];
        re = fma(w, c, re);
        im = fma(w, s, im);
    }
    T1[id] = make_double2(re, im);
}
// M(kx, ky) = sum_{rho_y} T1[c][rho_y][kx] e^{+2 pi i ky rho_y / L};  M' = M(kx + L/2, ky + L/2) (the (-1)^{rho_y} sum over
// the shifted column);  A = (M + M') / N,  B = (M - M') / N  at  AB[slot_x(kx)][slot_y(ky)],  kx < L/2.
__global__ void wq_pass2_kernel(const double2 *__restrict__ T1, float *__restrict__ AB, int L) {
    const int Lh = L >> 1;
    const size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= 4 * (size_t)Lh * L) return;
    const int kx = (int)(id % Lh), ky = (int)((id / Lh) % L), c = (int)(id / ((size_t)Lh * L));
    double re = 0.0, im = 0.0, re2 = 0.0, im2 = 0.0;
    for (int ry = 0; ry < L; ++ry) {
        double s, cs;
        sincospi(2.0 * (double)((ky * ry) % L) / (double)L, &s, &cs);
        const double2 a = T1[((size_t)c * L + ry) * L + kx], b = T1[((size_t)c * L + ry) * L + kx + Lh];
        const double sg = (ry & 1) ? -1.0 : 1.0;
        re += a.x * cs - a.y * s;
        im += a.x * s + a.y * cs;
        re2 += sg * (b.x * cs - b.y * s);
        im2 += sg * (b.x * s + b.y * cs);
    }
    const int N2 = L / 16, N2X = Lh >= 16 ? Lh / 16 : 1;
    const int sx = N2X * (kx & 15) + (kx >> 4), sy = N2 * (ky & 15) + (ky >> 4);
    const double inv = 1.0 / ((double)L * (double)L);
    // floats of one (slot_x, slot_y): Axx 0-1, Axy 2-3, Ayy 4-5, Bxx 6-7, Bxy 8-9, Byy 10-11, Azz 12-13, Bzz 14-15
    const int ia = c == 3 ? 12 : 2 * c, ib = c == 3 ? 14 : 6 + 2 * c;
    float *dst = AB + ((size_t)sx * L + sy) * 16;
    dst[ia] = (float)((re + re2) * inv);
    dst[ia + 1] = (float)((im + im2) * inv);
    dst[ib] = (float)((re - re2) * inv);
    dst[ib + 1] = (float)((im - im2) * inv);
}

// twf[j] = (c, -s), twi[j] = (c, s) with (c, s) = (cos, sin)(2 pi j / L), j < L, rounded from fp64
__global__ void twiddle_table_kernel(float2 *__restrict__ twf, float2 *__restrict__ twi, int L) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= L) return;
    double s, c;
    sincospi(2.0 * (double)j / (double)L, &s, &c);
    const float cf = (float)c, sf = (float)s;
    twf[j] = make_float2(cf, -sf);
    twi[j] = make_float2(cf, sf);
}

// The spins between the internal layout S[qc][a][P pairs] and the block-major copy SG[pb][qc][a][8 pairs] a chain of the
// branched replay works on (dsmc_api.cu: replay_sweep_graph).  One thread per replica pair of one site.
template <bool TO_BLOCKS>
__global__ void __launch_bounds__(256) spin_blocks_kernel(float2 *__restrict__ S, float2 *__restrict__ SG, size_t sites6, int P) {
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= sites6 * (size_t)P) return;
    const size_t qa = t / (size_t)P;                            // (qc, a) flattened: qc * Nh + a
    const int pair = (int)(t - qa * (size_t)P), pb = pair >> 3, ln = pair & 7;
    float2 *blk = SG + ((size_t)pb * sites6 + qa) * 8 + ln;
    if (TO_BLOCKS) *blk = S[t];
    else S[t] = *blk;
}

int pairs_per_cta(int P, int cap) {
    int ln = 1;
    while (ln * 2 <= cap && P % (ln * 2) == 0) ln *= 2;
    return ln;
}

template <int N2>
size_t y_smem_bytes(int LZ, int lines) {
    return sizeof(float2) * ((size_t)lines * 16 * N2 * LZ) + 2 * sizeof(float2) * 16 * N2 + 64;
}

template <int N2, int LZC>
cudaError_t launch_y(int mode, const FcParams &q, dim3 gy, dim3 by, size_t smy2, size_t smy4, cudaStream_t st) {
    if (mode == FC_FWD_ONLY) return launch_pdl(fftc_y_kernel<N2, FC_FWD_ONLY, LZC>, gy, by, smy2, st, q);
    if (mode == FC_FUSED) return launch_pdl(fftc_y_kernel<N2, FC_FUSED, LZC>, gy, by, smy4, st, q);
    return launch_pdl(fftc_y_kernel<N2, FC_COMBINE, LZC>, gy, by, smy4, st, q);
}

template <typename K>
cudaError_t raise_smem(K kern) { return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); }

// one field of colour `colour` (0 / 1), or of both (-1); valid[c] = "the cache holds the half-spectrum of colour c of the
// current spins" (kept by the caller across calls; a Metropolis update of colour c clears valid[c])
template <int N2X>
cudaError_t launch_row_update(const FcParams &q, const MetropolisArgs &ma, dim3 grid, dim3 block, size_t smem, cudaStream_t st) {
    const RoundKeys rk = make_round_keys(ma.seed_lo, ma.seed_hi);
    if (ma.step_dev && ma.flip) return launch_pdl(fftc_row_update_kernel<N2X, 8, true, 1>, grid, block, smem, st, q, ma, rk);
    if (ma.step_dev) return launch_pdl(fftc_row_update_kernel<N2X, 8, true, 0>, grid, block, smem, st, q, ma, rk);
    if (ma.flip) return launch_pdl(fftc_row_update_kernel<N2X, 8, false, 1>, grid, block, smem, st, q, ma, rk);
    return launch_pdl(fftc_row_update_kernel<N2X, 8, false, 0>, grid, block, smem, st, q, ma, rk);
}

// fuse != null (and colour 0 / 1): the x-inverse pass is replaced by the fused row kernel, which also takes the Metropolis
// decision of the half-sweep and leaves the forward-transformed rows of the updated colour in Z (*zline = that colour)
template <int N2>
cudaError_t launch_fftc(FcParams p, float2 *C, size_t cache_elems, int colour, bool *valid, int *zline, const MetropolisArgs *fuse,
                        int pb0, int npb, bool *configured, cudaStream_t st, uint64_t *launches) {
    constexpr int L = 16 * N2, N2X = N2 / 2 > 0 ? N2 / 2 : 1;
    static_assert(N2 >= 2, "L >= 32");
    // lines of 8 replica pairs (64-byte runs): four of them are 64 KB of shared memory at L = 256, three CTAs per SM
    int capz = 8;
    while (capz > 1 && y_smem_bytes<N2>(capz, 4) > 200 * 1024) capz >>= 1;
    p.LZ = pairs_per_cta(p.P, capz);
    p.PBZ = p.P / p.LZ;
    const int LNX = pairs_per_cta(p.P, 16);               // the x passes: 16 pairs per CTA = 128-byte runs of the spin arrays
    const bool fast = LNX == 16 && p.LZ == 8;             // lane counts known at compile time (config 5)
    const int TL = N2X < 16 ? N2X : 16;
    const size_t smx = sizeof(float2) * (L + (size_t)line_rows<N2X>() * LNX);
    const size_t smy2 = y_smem_bytes<N2>(p.LZ, 2), smy4 = y_smem_bytes<N2>(p.LZ, 4);
    if (!*configured) {
        cudaError_t e;
        if ((e = raise_smem(fftc_y_kernel<N2, FC_FWD_ONLY, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_y_kernel<N2, FC_FUSED, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_y_kernel<N2, FC_COMBINE, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_y_kernel<N2, FC_FWD_ONLY, 8>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_y_kernel<N2, FC_FUSED, 8>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_y_kernel<N2, FC_COMBINE, 8>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_x_forward_kernel<N2X, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_x_inverse_kernel<N2X, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_x_forward_kernel<N2X, 16>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_x_inverse_kernel<N2X, 16>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_row_update_kernel<N2X, 8, false, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_row_update_kernel<N2X, 8, false, 1>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_row_update_kernel<N2X, 8, true, 0>)) != cudaSuccess) return e;
        if ((e = raise_smem(fftc_row_update_kernel<N2X, 8, true, 1>)) != cudaSuccess) return e;
        *configured = true;
    }
    // npb > 0: only the line blocks pb0 .. pb0 + npb - 1 (16 replicas each).  Line blocks never exchange data, so a
    // running sweep can be cut into independent chains of launches (dsmc_api.cu: the branches of the sweep graph); the x
    // passes have no such cut, so this needs the running-sweep state (y pass FC_FUSED + fused row kernel only).
    const bool part = npb > 0 && !(pb0 == 0 && npb == p.PBZ);
    if (fuse && p.LZ != 8) return cudaErrorInvalidValue;    // the fused row kernel is built for lines of 8 pairs
    if (part) {
        const int tc = colour, oc = 1 - colour;
        if (!fuse || colour < 0 || pb0 < 0 || pb0 + npb > p.PBZ || !valid[tc] || valid[oc] || *zline != oc)
            return cudaErrorInvalidValue;
    }
    if (p.SG && !part) return cudaErrorInvalidValue;        // the block-major spins are the chains' business only
    if (part) {
        p.pb0 = pb0;
    } else {
        npb = p.PBZ;
    }
    const dim3 gx(p.P / LNX, L, 3), bx(LNX, TL), gy(npb, L / 2 + L / 4), by(p.LZ, 16, 2);
    cudaError_t e = cudaSuccess;
    auto x_forward = [&](int c) {
        FcParams q = p;
        q.colour = c;
        ++*launches;
        return fast ? launch_pdl(fftc_x_forward_kernel<N2X, 16>, gx, bx, smx, st, q)
                    : launch_pdl(fftc_x_forward_kernel<N2X, 0>, gx, bx, smx, st, q);
    };
    auto y_pass = [&](int mode, int c) {                   // c = the colour transformed forward / "new" colour
        FcParams q = p;
        q.colour = c;
        q.Cnew = C + (size_t)c * cache_elems;
        q.Ctgt = C + (size_t)(1 - c) * cache_elems;
        ++*launches;
        return fast ? launch_y<N2, 8>(mode, q, gy, by, smy2, smy4, st) : launch_y<N2, 0>(mode, q, gy, by, smy2, smy4, st);
    };
    auto x_inverse = [&](int c) {
        FcParams q = p;
        q.colour = c;
        ++*launches;
        return fast ? launch_pdl(fftc_x_inverse_kernel<N2X, 16>, gx, bx, smx, st, q)
                    : launch_pdl(fftc_x_inverse_kernel<N2X, 0>, gx, bx, smx, st, q);
    };
    for (int tc = 0; tc < 2 && e == cudaSuccess; ++tc) {
        if (colour >= 0 && colour != tc) continue;
        const int oc = 1 - tc;
        if (!valid[tc]) {                                  // the target colour's own half-spectrum is stale: refresh it alone
            if (*zline != tc && (e = x_forward(tc)) != cudaSuccess) break;
            if ((e = y_pass(FC_FWD_ONLY, tc)) != cudaSuccess) break;
            valid[tc] = true;
            *zline = -1;
        }
        if (!valid[oc]) {                                  // the running-sweep case: only the colour just updated is stale
            if (*zline != oc && (e = x_forward(oc)) != cudaSuccess) break;   // (the fused row kernel has left its lines in Z)
            if ((e = y_pass(FC_FUSED, oc)) != cudaSuccess) break;
            valid[oc] = true;
        } else {
            if ((e = y_pass(FC_COMBINE, oc)) != cudaSuccess) break;
        }
        *zline = -1;
        if (fuse) {
            FcParams q = p;
            q.colour = tc;
            ++*launches;
            const size_t smu = sizeof(float2) * (2 * L + 3 * (size_t)line_rows<N2X>() * p.LZ);
            e = launch_row_update<N2X>(q, *fuse, dim3(npb, L), dim3(p.LZ, TL, 3), smu, st);
            valid[tc] = false;                             // the spins of colour tc have changed ...
            *zline = tc;                                   // ... and their forward-transformed rows are in Z already
        } else {
            e = x_inverse(tc);
        }
    }
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace

bool dsmc_fft_supported(int L, int R) {
    return (R % 2 == 0) && (L == 32 || L == 64 || L == 128 || L == 256 || L == 512);
}
size_t dsmc_fft_m_floats(int L) { return 8 * (size_t)L * L + 4 * (size_t)L; }   // AB: (L/2) L slots of 16 floats; twf, twi
size_t dsmc_fft_cache_elems(int L, int R) { return 3 * (size_t)(L / 2) * L * (size_t)(R / 2); }   // float2 per colour
size_t dsmc_fft_scratch_bytes(int L, int R) {
    const size_t N = (size_t)L * L;
    const size_t z = sizeof(float2) * dsmc_fft_cache_elems(L, R), t1 = sizeof(double2) * 4 * N;
    return z > t1 ? z : t1;
}
size_t dsmc_fft_cache_bytes(int L, int R) { return 2 * sizeof(float2) * dsmc_fft_cache_elems(L, R); }

cudaError_t launch_make_fft_table(const float *Wc, float *AB, void *scratch, int L, cudaStream_t st, uint64_t *launches) {
    const size_t total = 4 * (size_t)L * L;
    wq_pass1_kernel<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(Wc, (double2 *)scratch, L);
    wq_pass2_kernel<<<(unsigned)((total / 2 + 127) / 128), 128, 0, st>>>((const double2 *)scratch, AB, L);
    float2 *tw = reinterpret_cast<float2 *>(AB + 8 * (size_t)L * L);
    twiddle_table_kernel<<<(L + 127) / 128, 128, 0, st>>>(tw, tw + L, L);
    *launches += 3;
    return cudaGetLastError();
}

bool dsmc_fft_fused_supported(int L, int R) { return dsmc_fft_supported(L, R) && R % 16 == 0; }
// line blocks (16 replicas each) of the fused path: the units a running sweep can be cut into (launch_field_fft: pb0, npb)
int dsmc_fft_line_blocks(int L, int R) { return dsmc_fft_fused_supported(L, R) ? R / 16 : 0; }

cudaError_t launch_spin_blocks(float *S, float *SG, int L, int R, bool to_blocks, cudaStream_t st, uint64_t *launches) {
    const size_t sites6 = 6 * (size_t)L * (L / 2), total = sites6 * (size_t)(R / 2);
    const unsigned grid = (unsigned)((total + 255) / 256);
    if (to_blocks) spin_blocks_kernel<true><<<grid, 256, 0, st>>>((float2 *)S, (float2 *)SG, sites6, R / 2);
    else spin_blocks_kernel<false><<<grid, 256, 0, st>>>((float2 *)S, (float2 *)SG, sites6, R / 2);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_field_fft(const float *S, const float *AB, void *scratch, void *cache, float *H, int L, int R, int colour,
                             bool *valid, int *zline, const MetropolisArgs *fuse, int pb0, int npb, float *SG, bool *configured,
                             cudaStream_t st, uint64_t *launches) {
    if (fuse && (colour < 0 || !dsmc_fft_fused_supported(L, R))) return cudaErrorInvalidValue;
    FcParams p;
    p.S = S;
    p.H = H;
    p.Z = (float2 *)scratch;
    p.Cnew = nullptr;
    p.Ctgt = nullptr;
    p.AB = (const float4 *)AB;
    p.twf = reinterpret_cast<const float2 *>(AB + 8 * (size_t)L * L);
    p.twi = p.twf + L;
    p.L = L;
    p.P = R / 2;
    p.LZ = 1;
    p.PBZ = 1;
    p.pb0 = 0;
    p.SG = SG;
    p.colour = 0;
    const size_t ce = dsmc_fft_cache_elems(L, R);
    switch (L / 16) {
        case 2: return launch_fftc<2>(p, (float2 *)cache, ce, colour, valid, zline, fuse, pb0, npb, configured, st, launches);
        case 4: return launch_fftc<4>(p, (float2 *)cache, ce, colour, valid, zline, fuse, pb0, npb, configured, st, launches);
        case 8: return launch_fftc<8>(p, (float2 *)cache, ce, colour, valid, zline, fuse, pb0, npb, configured, st, launches);
        case 16: return launch_fftc<16>(p, (float2 *)cache, ce, colour, valid, zline, fuse, pb0, npb, configured, st, launches);
        case 32: return launch_fftc<32>(p, (float2 *)cache, ce, colour, valid, zline, fuse, pb0, npb, configured, st, launches);
    }
    return cudaErrorInvalidValue;
}
