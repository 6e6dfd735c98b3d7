// field_fft.cu -- a1, spectral route ("more efficient
// parallelization of the dipole sum"): the dipole field as a batched circular convolution by FFT.
//
//   h_n^a = sum_m W^{ab}(m - n) s_m^b  =  (w' (*) s)(n),  w'(d) = W(-d)
//   => h^ = M . s^,   M^{ab}(k) = sum_rho W^{ab}(rho) e^{+i k.rho}
//
// W is real, so F^-1[ M F[a + i b] ] = w' (*) a + i w' (*) b for real fields a, b: two replicas ride
// through one complex transform as real and imaginary part.  In the [q][c][a][r] layout replicas
// r, r+1 are adjacent floats, i.e. the spin array already IS an array of complex "replica pairs";
// no packing, no Hermitian bookkeeping, and M may be complex (W need not be even).
//
// Three kernels per field, all fp32, every global access a contiguous run over replica pairs:
//   fft_x_forward   (row y, component c): gather the row from the two colour arrays, length-L FFT
//                    along x, write Z[c][y][slot_x][pair]
//   fft_y_multiply  (column slot_x, 16 pairs): FFT along y, multiply by M (mixing x and y
//                    components), inverse FFT along y, in place in Z
//   fft_x_inverse   (row y, component c): inverse FFT along x, scatter to H (only the colour asked)
// A length-L transform (L = 16 * N2, N2 in {2,...,32}) is the four-step algorithm: 16-point FFTs in
// registers over the stride-N2 sub-sequences, twiddle, one pass through shared memory, N2-point
// FFTs in registers.  The spectrum is left in "slot order" slot(k) = N2 * (k mod 16) + k div 16;
// the inverse runs the same steps backwards, so no bit/digit reversal pass exists anywhere and M
// is simply tabulated in slot order.  The 1/N of the inverse transform is folded into M.
#include "dsmc_internal.cuh"

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

// ---- the four steps of a length L = 16 * N2 transform --------------------------------------
// buf[sidx(k1, n2) * LN + lane] is the CTA's shared line buffer (LN = replica pairs per CTA): slot
// N2 k1 + n2 with one pad row per block of N2 slots, so that the two blocks a 16-lane warp touches in
// step 2 fall on different banks.  tw[j] = (cos, sin)(2 pi j / L).  Threads are (lane, t), t in [0, 16).
template <int N2>
__device__ __forceinline__ int sidx(int k1, int n2) { return (N2 + 1) * k1 + n2; }
template <int N2>
__host__ __device__ constexpr int line_rows() { return (N2 + 1) * 16; }

// forward step 1: v[n1] = x[N2 n1 + n2]  ->  A[k1][n2] * W_L^{n2 k1}  at slot N2 k1 + n2
template <int N2>
__device__ __forceinline__ void fwd_step1(float2 (&v)[16], int n2, const float2 *tw, float2 *buf, int LN, int lane) {
    fft_reg<16, false>(v);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const float2 w = tw[n2 * k1];
        buf[sidx<N2>(k1, n2) * LN + lane] = cmul(v[bitrev<16>(k1)], make_float2(w.x, -w.y));
    }
}
// forward step 2: the thread's block k1 -> u[k2] = X[k1 + 16 k2] in natural k2 order
template <int N2>
__device__ __forceinline__ void fwd_step2(float2 (&u)[N2], int k1, const float2 *buf, int LN, int lane) {
    float2 t[N2];
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2) t[n2] = buf[sidx<N2>(k1, n2) * LN + lane];
    fft_reg<N2, false>(t);
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) u[k2] = t[bitrev<N2>(k2)];
}
// inverse step 2: u[k2] = Y[k1 + 16 k2]  ->  B[k1][n2] * conj(W_L^{n2 k1})  at slot N2 k1 + n2
template <int N2>
__device__ __forceinline__ void inv_step2(float2 (&u)[N2], int k1, const float2 *tw, float2 *buf, int LN, int lane) {
    fft_reg<N2, true>(u);
#pragma unroll
    for (int n2 = 0; n2 < N2; ++n2) buf[sidx<N2>(k1, n2) * LN + lane] = cmul(u[bitrev<N2>(n2)], tw[n2 * k1]);
}
// inverse step 1: slots N2 k1 + n2 (k1 = 0..15)  ->  v[n1] = x[N2 n1 + n2]
template <int N2>
__device__ __forceinline__ void inv_step1(float2 (&v)[16], int n2, const float2 *buf, int LN, int lane) {
    float2 t[16];
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) t[k1] = buf[sidx<N2>(k1, n2) * LN + lane];
    fft_reg<16, true>(t);
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) v[n1] = t[bitrev<16>(n1)];
}

__device__ __forceinline__ void fill_twiddles(float2 *tw, int L) {
    const int tid = threadIdx.y * blockDim.x + threadIdx.x, nt = blockDim.x * blockDim.y;
    for (int j = tid; j < L; j += nt) {
        float s, c;
        sincospif(2.0f * (float)j / (float)L, &s, &c);   // exact argument: j / L is a dyadic fraction
        tw[j] = make_float2(c, s);
    }
}

struct FftParams {
    const float *S;   // spins, internal layout
    float *H;         // field, internal layout
    float2 *Z;        // spectrum scratch Z[c][y][slot_x][pair]
    const float4 *M;  // M[slot_x][slot_y][2]: (xx.re, xx.im, xy.re, xy.im), (yy.re, yy.im, zz.re, zz.im), scaled 1/N
    int L, P;         // P = R / 2 complex replica pairs
    int colour;       // which targets fft_x_inverse writes: -1 both colours, 0, 1
};

// grid (P / LN, L, 3), block (LN, 16)
template <int N2>
__global__ void __launch_bounds__(512) fft_x_forward_kernel(const FftParams p) {
    extern __shared__ __align__(16) float2 fsm[];
    const int L = 16 * N2, Lh = L / 2, LN = blockDim.x;
    float2 *tw = fsm, *buf = fsm + L;
    const int lane = threadIdx.x, t = threadIdx.y;
    const int pair = blockIdx.x * LN + lane, y = blockIdx.y, c = blockIdx.z;
    const size_t planeP = (size_t)L * Lh * p.P;
    const float2 *S2 = reinterpret_cast<const float2 *>(p.S);
    auto load_line = [&](float2 (&v)[16], int n2) {
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const int x = N2 * n1 + n2, q = (x + y) & 1;
            v[n1] = __ldg(S2 + (size_t)(q * 3 + c) * planeP + (size_t)(y * Lh + (x >> 1)) * p.P + pair);
        }
    };
    // the twiddles do not depend on the spins: they are computed while the kernel that writes the spins may still run
    // the first sub-sequence's loads are issued before the twiddles are computed: they do not depend on them
    pdl_wait();                                            // the spins come from the Metropolis kernel before
    float2 v0[16];
    if (t < N2) load_line(v0, t);
    fill_twiddles(tw, L);
    __syncthreads();
    if (t < N2) fwd_step1<N2>(v0, t, tw, buf, LN, lane);
    for (int n2 = t + 16; n2 < N2; n2 += 16) {
        float2 v[16];
        load_line(v, n2);
        fwd_step1<N2>(v, n2, tw, buf, LN, lane);
    }
    __syncthreads();
    pdl_trigger();                                         // late: a successor resident earlier only takes room (section 5.2b)
    float2 u[N2];
    fwd_step2<N2>(u, t, buf, LN, lane);
    float2 *dst = p.Z + ((size_t)(c * L + y) * L + N2 * t) * p.P + pair;
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) dst[(size_t)k2 * p.P] = u[k2];
}

// grid (P / LN, L, 3), block (LN, 16)
template <int N2>
__global__ void __launch_bounds__(512) fft_x_inverse_kernel(const FftParams p) {
    extern __shared__ __align__(16) float2 fsm[];
    const int L = 16 * N2, Lh = L / 2, LN = blockDim.x;
    float2 *tw = fsm, *buf = fsm + L;
    const int lane = threadIdx.x, t = threadIdx.y;
    const int pair = blockIdx.x * LN + lane, y = blockIdx.y, c = blockIdx.z;
    float2 u[N2];
    const float2 *src = p.Z + ((size_t)(c * L + y) * L + N2 * t) * p.P + pair;
    pdl_wait();                                            // the spectrum comes from the y pass
#pragma unroll
    for (int k2 = 0; k2 < N2; ++k2) u[k2] = src[(size_t)k2 * p.P];
    fill_twiddles(tw, L);
    __syncthreads();
    bool folded = false;
    if constexpr (N2 == 16) {
        // One colour wanted: of the N2 outputs n2 of inverse step 2 only those of parity par = (colour + y) & 1 are
        // used below, so the step is an 8-point transform of the folded input (the same radix-2 step by hand as in the
        // last step; par is uniform over the CTA)
        if (p.colour >= 0) {
            const int par = (p.colour + y) & 1;
            float2 a[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (par) {
                    const float2 d = csub(u[k], u[k + 8]);
                    a[k] = k == 0 ? d : k == 4 ? make_float2(-d.y, d.x) : cmul(d, make_float2(kTw32.c[2 * k], kTw32.s[2 * k]));
                } else {
                    a[k] = cadd(u[k], u[k + 8]);
                }
            }
            fft_reg<8, true>(a);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int n2 = par + 2 * j;
                buf[sidx<N2>(t, n2) * LN + lane] = cmul(a[bitrev<8>(j)], tw[n2 * t]);
            }
            folded = true;
        }
    }
    if (!folded) inv_step2<N2>(u, t, tw, buf, LN, lane);
    pdl_trigger();
    __syncthreads();
    const size_t planeP = (size_t)L * Lh * p.P;
    float2 *H2 = reinterpret_cast<float2 *>(p.H);
    if constexpr (N2 == 16) {
        // One colour wanted: only the 8 sub-sequences n2 of the right parity are transformed, which would leave every
        // second t idle.  Instead the 16 t share them in pairs, t < 8 taking the even and t >= 8 the odd outputs n1 of
        // sub-sequence n2 = par + 2 (t & 7) (a warp holds two consecutive t, so neither half diverges): one radix-2
        // step by hand, x[2j] = F8^-1[t_k + t_{k+8}](j), x[2j+1] = F8^-1[(t_k - t_{k+8}) w^k](j), w = e^{2 pi i / 16}.
        if (p.colour >= 0) {
            const int par = (p.colour + y) & 1, n2 = par + 2 * (t & 7), odd = t >> 3;
            float2 a[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const float2 lo = buf[sidx<N2>(k, n2) * LN + lane], hi = buf[sidx<N2>(k + 8, n2) * LN + lane];
                if (odd) {
                    const float2 d = csub(lo, hi);
                    a[k] = k == 0 ? d : k == 4 ? make_float2(-d.y, d.x) : cmul(d, make_float2(kTw32.c[2 * k], kTw32.s[2 * k]));
                } else {
                    a[k] = cadd(lo, hi);
                }
            }
            fft_reg<8, true>(a);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int x = N2 * (2 * j + odd) + n2;                 // parity of n2: colour p.colour
                H2[(size_t)(p.colour * 3 + c) * planeP + (size_t)(y * Lh + (x >> 1)) * p.P + pair] = a[bitrev<8>(j)];
            }
            return;
        }
    }
    for (int n2 = t; n2 < N2; n2 += 16) {
        if (p.colour >= 0 && ((n2 + y) & 1) != p.colour) continue;   // x = N2 n1 + n2 has the parity of n2
        float2 v[16];
        inv_step1<N2>(v, n2, buf, LN, lane);
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) {
            const int x = N2 * n1 + n2, q = (x + y) & 1;
            H2[(size_t)(q * 3 + c) * planeP + (size_t)(y * Lh + (x >> 1)) * p.P + pair] = v[n1];
        }
    }
}

__device__ __forceinline__ float2 cmac(float2 acc, float2 a, float2 m) {  // acc + a * m
    return make_float2(fmaf(a.x, m.x, fmaf(-a.y, m.y, acc.x)), fmaf(a.x, m.y, fmaf(a.y, m.x, acc.y)));
}

// grid (P / LN, L slots), block (LN, 16); shared: twiddles + 3 line buffers
template <int N2>
__global__ void __launch_bounds__(256, 2) fft_y_multiply_kernel(const FftParams p) {
    extern __shared__ __align__(16) float2 fsm[];
    const int L = 16 * N2, LN = blockDim.x;
    float2 *tw = fsm;
    float4 *Msm = reinterpret_cast<float4 *>(fsm + L);     // this column's multiplier, 2 float4 per slot_y
    float2 *b0 = fsm + L + 4 * L;
    float2 *buf[3] = {b0, b0 + (size_t)line_rows<N2>() * LN, b0 + 2 * (size_t)line_rows<N2>() * LN};
    const int lane = threadIdx.x, t = threadIdx.y;
    const int pair = blockIdx.x * LN + lane, sx = blockIdx.y;
    fill_twiddles(tw, L);
    for (int j = t * LN + lane; j < 2 * L; j += 16 * LN) Msm[j] = __ldg(p.M + (size_t)sx * L * 2 + j);  // constant table
    pdl_wait();                                            // the spectrum comes from the x pass
    __syncthreads();
    const size_t rowP = (size_t)L * p.P;                   // one y step in Z
    float2 *col = p.Z + (size_t)sx * p.P + pair;           // + (c * L + y) * rowP
#pragma unroll 1
    for (int c = 0; c < 3; ++c)
        for (int n2 = t; n2 < N2; n2 += 16) {
            float2 v[16];
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) v[n1] = col[(size_t)(c * L + N2 * n1 + n2) * rowP];
            fwd_step1<N2>(v, n2, tw, buf[c], LN, lane);
        }
    __syncthreads();
    {
        const float4 *Mrow = Msm + (N2 * t) * 2;
        // The thread owns block t of all three components, so the x spectrum can wait in its own
        // shared-memory block (natural k2 order) while the y spectrum is transformed: at most one
        // block lives in registers at a time.
        float2 ux[N2];
        float2 *bx = buf[0] + sidx<N2>(t, 0) * LN + lane;
        fwd_step2<N2>(ux, t, buf[0], LN, lane);
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) bx[k2 * LN] = ux[k2];
        fwd_step2<N2>(ux, t, buf[1], LN, lane);            // ux now holds the y component
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) {
            const float4 m0 = Mrow[2 * k2], m1 = Mrow[2 * k2 + 1];
            const float2 xx = make_float2(m0.x, m0.y), xy = make_float2(m0.z, m0.w), yy = make_float2(m1.x, m1.y);
            const float2 zx = bx[k2 * LN], zy = ux[k2];
            bx[k2 * LN] = cmac(cmul(zx, xx), zy, xy);
            ux[k2] = cmac(cmul(zx, xy), zy, yy);
        }
        inv_step2<N2>(ux, t, tw, buf[1], LN, lane);
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) ux[k2] = bx[k2 * LN];
        inv_step2<N2>(ux, t, tw, buf[0], LN, lane);
        fwd_step2<N2>(ux, t, buf[2], LN, lane);            // ux reused for the z component
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) {
            const float4 m1 = Mrow[2 * k2 + 1];
            ux[k2] = cmul(ux[k2], make_float2(m1.z, m1.w));
        }
        inv_step2<N2>(ux, t, tw, buf[2], LN, lane);
    }
    __syncthreads();
    pdl_trigger();
#pragma unroll 1
    for (int c = 0; c < 3; ++c)
        for (int n2 = t; n2 < N2; n2 += 16) {
            float2 v[16];
            inv_step1<N2>(v, n2, buf[c], LN, lane);
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) col[(size_t)(c * L + N2 * n1 + n2) * rowP] = v[n1];
        }
}

// ---- M = transform of W, fp64, once per tensor ------------------------------------------------
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
// M[slot(kx)][slot(ky)][c] = (1/N) sum_{rho_y} T1[c][rho_y][kx] e^{+2 pi i ky rho_y / L}
__global__ void wq_pass2_kernel(const double2 *__restrict__ T1, float *__restrict__ M, int L) {
    const size_t N = (size_t)L * L;
    const size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= 4 * N) return;
    const int kx = (int)(id % L), ky = (int)((id / L) % L), c = (int)(id / N);
    double re = 0.0, im = 0.0;
    for (int ry = 0; ry < L; ++ry) {
        double s, cs;
        sincospi(2.0 * (double)((ky * ry) % L) / (double)L, &s, &cs);
        const double2 t = T1[((size_t)c * L + ry) * L + kx];
        re += t.x * cs - t.y * s;
        im += t.x * s + t.y * cs;
    }
    const int N2 = L / 16;
    const int sx = N2 * (kx & 15) + (kx >> 4), sy = N2 * (ky & 15) + (ky >> 4);
    float *dst = M + ((size_t)sx * L + sy) * 8 + 2 * c;
    dst[0] = (float)(re / (double)N);
    dst[1] = (float)(im / (double)N);
}

int pairs_per_cta(int P, int cap) {
    int ln = 1;
    while (ln * 2 <= cap && P % (ln * 2) == 0) ln *= 2;
    return ln;
}

template <int N2>
cudaError_t launch_fft_n2(const FftParams &p, bool *configured, cudaStream_t st, uint64_t *launches) {
    const int L = 16 * N2;
    // 16 replica pairs per CTA: 128-byte runs in HBM, and enough CTAs (half rows / half columns) that
    // the last wave over 148 SMs stays full
    const int LNX = pairs_per_cta(p.P, 16), LNY = pairs_per_cta(p.P, 16);
    const size_t smx = sizeof(float2) * (L + (size_t)line_rows<N2>() * LNX);
    const size_t smy = sizeof(float2) * (L + 4 * L + 3 * (size_t)line_rows<N2>() * LNY);
    if (!*configured) {
        cudaError_t e;
        if ((e = cudaFuncSetAttribute(fft_x_forward_kernel<N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(fft_x_inverse_kernel<N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(fft_y_multiply_kernel<N2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024)) != cudaSuccess) return e;
        *configured = true;
    }
    cudaError_t e = launch_pdl(fft_x_forward_kernel<N2>, dim3(p.P / LNX, L, 3), dim3(LNX, 16), smx, st, p);
    if (e == cudaSuccess) e = launch_pdl(fft_y_multiply_kernel<N2>, dim3(p.P / LNY, L), dim3(LNY, 16), smy, st, p);
    if (e == cudaSuccess) e = launch_pdl(fft_x_inverse_kernel<N2>, dim3(p.P / LNX, L, 3), dim3(LNX, 16), smx, st, p);
    *launches += 3;
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace

bool dsmc_fft_supported(int L, int R) {
    return (R % 2 == 0) && (L == 32 || L == 64 || L == 128 || L == 256 || L == 512);
}
size_t dsmc_fft_m_floats(int L) { return 8 * (size_t)L * L; }
size_t dsmc_fft_scratch_bytes(int L, int R) {
    const size_t N = (size_t)L * L;
    const size_t z = sizeof(float) * 3 * N * R, t1 = sizeof(double2) * 4 * N;
    return z > t1 ? z : t1;
}

cudaError_t launch_make_fft_table(const float *Wc, float *M, void *scratch, int L, cudaStream_t st, uint64_t *launches) {
    const size_t total = 4 * (size_t)L * L;
    const unsigned grid = (unsigned)((total + 127) / 128);
    wq_pass1_kernel<<<grid, 128, 0, st>>>(Wc, (double2 *)scratch, L);
    wq_pass2_kernel<<<grid, 128, 0, st>>>((const double2 *)scratch, M, L);
    *launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_field_fft(const float *S, const float *M, void *scratch, float *H, int L, int R, int colour,
                             bool *configured, cudaStream_t st, uint64_t *launches) {
    FftParams p;
    p.S = S;
    p.H = H;
    p.Z = (float2 *)scratch;
    p.M = (const float4 *)M;
    p.L = L;
    p.P = R / 2;
    p.colour = colour;
    switch (L / 16) {
        case 2: return launch_fft_n2<2>(p, configured, st, launches);
        case 4: return launch_fft_n2<4>(p, configured, st, launches);
        case 8: return launch_fft_n2<8>(p, configured, st, launches);
        case 16: return launch_fft_n2<16>(p, configured, st, launches);
        case 32: return launch_fft_n2<32>(p, configured, st, launches);
    }
    return cudaErrorInvalidValue;
}
