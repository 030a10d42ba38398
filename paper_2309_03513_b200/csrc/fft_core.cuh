// Mixed-radix (2,3,5) FP64 FFT core: register butterflies and an in-place multi-stage transform on a
// shared-memory tile.  Forward = decimation in frequency (natural order in, digit-reversed order out),
// inverse = decimation in time (digit-reversed in, natural out), so no reordering pass is ever needed:
// every frequency-space array of the library lives in the digit-reversed ("scrambled") order and the
// host tables (Coulomb kernel, sphere index maps) are built in that order (plan.cpp).
//
// The paper asks only for "fast Fourier transforms (FFTs) between the direct and reciprocal spaces"
// (PAPER.md:274); the design here is B200-first: radix-8/9/10 butterflies in registers (FP64 issue is the
// scarce resource, 64 DFMA/clk/SM measured), tiles staged in shared memory, conflict-free 16-byte lanes.
//
// The core is __host__ __device__ so the host unit tests can run the very same index logic.
#pragma once
#include <cuda_runtime.h>

namespace tddft {

typedef double2 cplx;

#define TD_HD __host__ __device__ __forceinline__

// ---------------------------------------------------------------------------------------------------
// compile-time trigonometry: cos/sin(2 pi j / n) evaluated by the host front end in long double
namespace ct {
constexpr long double PI_L = 3.14159265358979323846264338327950288L;
constexpr long double sin_series(long double x) {   // |x| <= pi/4
    long double term = x, sum = x, x2 = x * x;
    for (int k = 1; k < 16; ++k) { term *= -x2 / ((2 * k) * (2 * k + 1)); sum += term; }
    return sum;
}
constexpr long double cos_series(long double x) {   // |x| <= pi/4
    long double term = 1, sum = 1, x2 = x * x;
    for (int k = 1; k < 16; ++k) { term *= -x2 / ((2 * k - 1) * (2 * k)); sum += term; }
    return sum;
}
// cos(2 pi a / m) for integers, exact octant reduction on the rational a/m
constexpr long double cos2pi(long long a, long long m) {
    a %= m; if (a < 0) a += m;
    if (2 * a > m) a = m - a;                       // cos is even about pi
    if (4 * a > m) return -cos2pi(m - 2 * a, 2 * m);  // cos(x) = -cos(pi - x); pi - x = 2 pi (m - 2a)/(2m)
    // now 0 <= a/m <= 1/4
    if (8 * a <= m) return cos_series(2 * PI_L * a / m);
    return sin_series(2 * PI_L * (m - 4 * a) / (4 * m));   // cos(x) = sin(pi/2 - x)
}
constexpr long double sin2pi(long long a, long long m) { return cos2pi(4 * a - m, 4 * m); }  // sin(x) = cos(x - pi/2)
}  // namespace ct

template <int N, int J> struct Tw {   // exp(-2 pi i J / N)
    static constexpr double c = (double)ct::cos2pi(J, N);
    static constexpr double s = -(double)ct::sin2pi(J, N);
};

template <int I> struct IC { static constexpr int value = I; };
template <int B, int E, class F> TD_HD void static_for(F&& f) {
    if constexpr (B < E) { f(IC<B>{}); static_for<B + 1, E>(f); }
}

TD_HD cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
TD_HD cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
TD_HD cplx cmul(cplx a, cplx b) { return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x)); }
TD_HD cplx cmulc(cplx a, cplx b) { return make_double2(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -a.x * b.y)); }  // a * conj(b)
template <bool INV> TD_HD cplx mul_mi(cplx a) {   // forward: a * (-i); inverse: a * (+i)
    return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x);
}
template <bool INV, int N, int J> TD_HD cplx mul_tw(cplx a) {   // a * exp(-/+ 2 pi i J / N) with literal constants
    constexpr int j = ((J % N) + N) % N;
    if constexpr (j == 0) return a;
    else if constexpr (4 * j == N) return mul_mi<INV>(a);
    else if constexpr (2 * j == N) return make_double2(-a.x, -a.y);
    else if constexpr (4 * j == 3 * N) return mul_mi<!INV>(a);
    else {
        constexpr double c = Tw<N, j>::c;
        constexpr double s = INV ? -Tw<N, j>::s : Tw<N, j>::s;
        return make_double2(fma(a.x, c, -a.y * s), fma(a.x, s, a.y * c));
    }
}

// ---------------------------------------------------------------------------------------------------
// radix-R butterflies on registers: X[k] = sum_n x[n] exp(-/+ 2 pi i n k / R), natural order in and out
template <int R, bool INV> struct Dft;

template <bool INV> struct Dft<2, INV> {
    static TD_HD void run(cplx (&x)[2]) { cplx a = x[0], b = x[1]; x[0] = cadd(a, b); x[1] = csub(a, b); }
};
template <bool INV> struct Dft<3, INV> {
    static TD_HD void run(cplx (&x)[3]) {
        constexpr double s = INV ? -0.86602540378443864676 : 0.86602540378443864676;   // sin(2 pi/3), sign of -i
        cplx t1 = cadd(x[1], x[2]);
        cplx t2 = make_double2(fma(-0.5, t1.x, x[0].x), fma(-0.5, t1.y, x[0].y));
        cplx d = csub(x[1], x[2]);
        cplx t3 = make_double2(s * d.y, -s * d.x);        // forward: -i s d
        x[0] = cadd(x[0], t1); x[1] = cadd(t2, t3); x[2] = csub(t2, t3);
    }
};
template <bool INV> struct Dft<4, INV> {
    static TD_HD void run(cplx (&x)[4]) {
        cplx t0 = cadd(x[0], x[2]), t1 = csub(x[0], x[2]), t2 = cadd(x[1], x[3]), t3 = mul_mi<INV>(csub(x[1], x[3]));
        x[0] = cadd(t0, t2); x[1] = cadd(t1, t3); x[2] = csub(t0, t2); x[3] = csub(t1, t3);
    }
};
template <bool INV> struct Dft<5, INV> {
    static TD_HD void run(cplx (&x)[5]) {
        constexpr double c1 = Tw<5, 1>::c, c2 = Tw<5, 2>::c;
        constexpr double s1 = INV ? Tw<5, 1>::s : -Tw<5, 1>::s;     // +sin(2 pi/5) forward
        constexpr double s2 = INV ? Tw<5, 2>::s : -Tw<5, 2>::s;
        cplx a1 = cadd(x[1], x[4]), a2 = cadd(x[2], x[3]), b1 = csub(x[1], x[4]), b2 = csub(x[2], x[3]);
        cplx p1 = make_double2(fma(c2, a2.x, fma(c1, a1.x, x[0].x)), fma(c2, a2.y, fma(c1, a1.y, x[0].y)));
        cplx p2 = make_double2(fma(c1, a2.x, fma(c2, a1.x, x[0].x)), fma(c1, a2.y, fma(c2, a1.y, x[0].y)));
        cplx q1 = make_double2(fma(s2, b2.x, s1 * b1.x), fma(s2, b2.y, s1 * b1.y));
        cplx q2 = make_double2(fma(-s1, b2.x, s2 * b1.x), fma(-s1, b2.y, s2 * b1.y));
        // forward: X1 = p1 - i q1, X4 = p1 + i q1, X2 = p2 - i q2, X3 = p2 + i q2 (s carries the sign for the inverse)
        x[0] = cadd(x[0], cadd(a1, a2));
        x[1] = make_double2(p1.x + q1.y, p1.y - q1.x);
        x[4] = make_double2(p1.x - q1.y, p1.y + q1.x);
        x[2] = make_double2(p2.x + q2.y, p2.y - q2.x);
        x[3] = make_double2(p2.x - q2.y, p2.y + q2.x);
    }
};
// composite R = RA * RB: Cooley-Tukey inside registers, constants folded at compile time
template <int RA, int RB, bool INV> struct DftComposite {
    static constexpr int R = RA * RB;
    static TD_HD void run(cplx (&x)[R]) {
        cplx t[R];
        static_for<0, RB>([&](auto nb_) {
            constexpr int nb = decltype(nb_)::value;
            cplx y[RA];
            static_for<0, RA>([&](auto na_) { constexpr int na = decltype(na_)::value; y[na] = x[na * RB + nb]; });
            Dft<RA, INV>::run(y);
            static_for<0, RA>([&](auto ka_) {
                constexpr int ka = decltype(ka_)::value;
                t[ka * RB + nb] = mul_tw<INV, R, nb * ka>(y[ka]);
            });
        });
        static_for<0, RA>([&](auto ka_) {
            constexpr int ka = decltype(ka_)::value;
            cplx z[RB];
            static_for<0, RB>([&](auto nb_) { constexpr int nb = decltype(nb_)::value; z[nb] = t[ka * RB + nb]; });
            Dft<RB, INV>::run(z);
            static_for<0, RB>([&](auto kb_) { constexpr int kb = decltype(kb_)::value; x[ka + RA * kb] = z[kb]; });
        });
    }
};
template <bool INV> struct Dft<6, INV> { static TD_HD void run(cplx (&x)[6]) { DftComposite<2, 3, INV>::run(x); } };
template <bool INV> struct Dft<8, INV> { static TD_HD void run(cplx (&x)[8]) { DftComposite<2, 4, INV>::run(x); } };
template <bool INV> struct Dft<9, INV> { static TD_HD void run(cplx (&x)[9]) { DftComposite<3, 3, INV>::run(x); } };
template <bool INV> struct Dft<10, INV> { static TD_HD void run(cplx (&x)[10]) { DftComposite<2, 5, INV>::run(x); } };
template <bool INV> struct Dft<12, INV> { static TD_HD void run(cplx (&x)[12]) { DftComposite<3, 4, INV>::run(x); } };
template <bool INV> struct Dft<15, INV> { static TD_HD void run(cplx (&x)[15]) { DftComposite<3, 5, INV>::run(x); } };
template <bool INV> struct Dft<16, INV> { static TD_HD void run(cplx (&x)[16]) { DftComposite<4, 4, INV>::run(x); } };

// ---------------------------------------------------------------------------------------------------
// plans: N = R1 * R2 * R3 (R = 1 means "no stage").  Forward runs R1 first on the full length.
template <int N> struct Plan;
#define TD_PLAN(N_, A_, B_, C_) template <> struct Plan<N_> { static constexpr int R1 = A_, R2 = B_, R3 = C_; };
TD_PLAN(4, 4, 1, 1)    TD_PLAN(5, 5, 1, 1)    TD_PLAN(6, 6, 1, 1)    TD_PLAN(8, 8, 1, 1)    TD_PLAN(9, 9, 1, 1)
TD_PLAN(10, 10, 1, 1)  TD_PLAN(12, 3, 4, 1)   TD_PLAN(15, 5, 3, 1)   TD_PLAN(16, 4, 4, 1)   TD_PLAN(18, 3, 6, 1)
TD_PLAN(20, 5, 4, 1)   TD_PLAN(24, 6, 4, 1)   TD_PLAN(25, 5, 5, 1)   TD_PLAN(27, 3, 9, 1)   TD_PLAN(30, 5, 6, 1)
TD_PLAN(32, 8, 4, 1)   TD_PLAN(36, 6, 6, 1)   TD_PLAN(40, 5, 8, 1)   TD_PLAN(45, 5, 9, 1)   TD_PLAN(48, 6, 8, 1)
TD_PLAN(50, 5, 10, 1)  TD_PLAN(54, 9, 6, 1)   TD_PLAN(60, 10, 6, 1)  TD_PLAN(64, 8, 8, 1)   TD_PLAN(72, 9, 8, 1)
TD_PLAN(75, 5, 5, 3)   TD_PLAN(80, 10, 8, 1)  TD_PLAN(81, 9, 9, 1)   TD_PLAN(90, 9, 10, 1)  TD_PLAN(96, 12, 8, 1)
TD_PLAN(100, 10, 10, 1) TD_PLAN(108, 12, 9, 1) TD_PLAN(120, 5, 6, 4)  TD_PLAN(125, 5, 5, 5)  TD_PLAN(128, 16, 8, 1)
TD_PLAN(144, 9, 4, 4)  TD_PLAN(150, 5, 5, 6)  TD_PLAN(160, 10, 4, 4) TD_PLAN(180, 5, 6, 6)  TD_PLAN(192, 6, 8, 4)
TD_PLAN(200, 5, 10, 4) TD_PLAN(216, 6, 6, 6)  TD_PLAN(240, 10, 6, 4) TD_PLAN(250, 5, 5, 10) TD_PLAN(256, 8, 8, 4)
#undef TD_PLAN
// the sizes the host dispatch instantiates
#define TD_FOR_EACH_N(X) X(4) X(5) X(6) X(8) X(9) X(10) X(12) X(15) X(16) X(18) X(20) X(24) X(25) X(27) X(30) X(32) X(36) X(40) \
    X(45) X(48) X(50) X(54) X(60) X(64) X(72) X(75) X(80) X(81) X(90) X(96) X(100) X(108) X(120) X(125) X(128) X(144) X(150)  \
    X(160) X(180) X(192) X(200) X(216) X(240) X(250) X(256)

template <int N> struct PlanInfo {
    static constexpr int R1 = Plan<N>::R1, R2 = Plan<N>::R2, R3 = Plan<N>::R3;
    static constexpr int NST = (R2 == 1) ? 1 : (R3 == 1 ? 2 : 3);
    static constexpr int RLAST = (NST == 1) ? R1 : (NST == 2 ? R2 : R3);
    // "along" tiles pad one element every RLAST elements when RLAST is even (conflict-free last stage)
    static constexpr int PADP = (RLAST % 2 == 0) ? RLAST : 0;
    static constexpr int NPAD = PADP ? N + N / PADP : N;
    static constexpr int MAXR = (R1 > R2 ? (R1 > R3 ? R1 : R3) : (R2 > R3 ? R2 : R3));
    static constexpr int MINR = NST == 1 ? R1 : (NST == 2 ? (R1 < R2 ? R1 : R2) : (R1 < R2 ? (R1 < R3 ? R1 : R3) : (R2 < R3 ? R2 : R3)));
    static constexpr int MAXJ = N / MINR;    // most butterflies per pencil in any stage
};
template <int N> TD_HD int pad_pos(int e) {
    if constexpr (PlanInfo<N>::PADP != 0) return e + e / PlanInfo<N>::PADP; else return e;
}

// One stage of radix R on blocks of length L (sub-stride L/R) for P pencils of a tile.
// ALONG: pencils are contiguous runs (element stride 1, padded), lanes run along the pencil.
// !ALONG: element stride = estride, pencil stride 1, lanes run across pencils.
// tw[k] = exp(-2 pi i k / N).
template <int N, int R, int L, bool INV, bool ALONG>
TD_HD void fft_stage(cplx* s, int P, int pstride, int estride, const cplx* tw, int tid, int nthr) {
    constexpr int ST = L / R;
    constexpr int J = N / R;
    const int items = P * J;
    for (int t = tid; t < items; t += nthr) {
        int p, j;
        if (ALONG) { p = t / J; j = t - p * J; } else { j = t / P; p = t - j * P; }
        const int blk = j / ST, i = j - blk * ST;
        const int e0 = blk * L + i;
        cplx x[R];
        cplx* base = s + (ALONG ? p * pstride : p);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int e = e0 + r * ST;
            x[r] = base[ALONG ? pad_pos<N>(e) : e * estride];
        }
        if (INV && ST > 1) {
#pragma unroll
            for (int r = 1; r < R; ++r) x[r] = cmulc(x[r], tw[i * r * (N / L)]);
        }
        Dft<R, INV>::run(x);
        if (!INV && ST > 1) {
#pragma unroll
            for (int r = 1; r < R; ++r) x[r] = cmul(x[r], tw[i * r * (N / L)]);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int e = e0 + r * ST;
            base[ALONG ? pad_pos<N>(e) : e * estride] = x[r];
        }
    }
}

// host-side mirror of the output order: freq_at_pos[p] = frequency index stored at position p after the forward DIF
inline void scrambled_order(int N, int R1, int R2, int R3, int* freq_at_pos) {
    int radices[3] = {R1, R2, R3};
    // recursive definition unrolled: position p = k1*(N/R1) + p', frequency k = R1*k' + k1
    struct Rec {
        static void go(int n, const int* r, int nr, int* out) {
            if (nr == 0 || n == 1) { out[0] = 0; return; }
            int R = r[0], M = n / R;
            int* sub = new int[M];
            go(M, r + 1, nr - 1, sub);
            for (int k1 = 0; k1 < R; ++k1) for (int p = 0; p < M; ++p) out[k1 * M + p] = R * sub[p] + k1;
            delete[] sub;
        }
    };
    int nr = (R2 == 1) ? 1 : (R3 == 1 ? 2 : 3);
    Rec::go(N, radices, nr, freq_at_pos);
}

}  // namespace tddft

namespace tddft {

struct NoSync { TD_HD void operator()() const {} };
struct BlockSync {
    TD_HD void operator()() const {
#ifdef __CUDA_ARCH__
        __syncthreads();
#endif
    }
};

// Full in-place transform of a tile: forward (DIF) or inverse (DIT, unnormalised).
// SYNC is called between stages (device: __syncthreads; host tests: nothing).
template <int N, bool INV, bool ALONG, class Sync>
TD_HD void fft_tile(cplx* s, int P, int pstride, int estride, const cplx* tw, int tid, int nthr, Sync sync) {
    using PI = PlanInfo<N>;
    constexpr int R1 = PI::R1, R2 = PI::R2, R3 = PI::R3;
    if constexpr (!INV) {
        fft_stage<N, R1, N, false, ALONG>(s, P, pstride, estride, tw, tid, nthr);
        if constexpr (PI::NST >= 2) { sync(); fft_stage<N, R2, N / R1, false, ALONG>(s, P, pstride, estride, tw, tid, nthr); }
        if constexpr (PI::NST >= 3) { sync(); fft_stage<N, R3, N / (R1 * R2), false, ALONG>(s, P, pstride, estride, tw, tid, nthr); }
    } else {
        if constexpr (PI::NST >= 3) { fft_stage<N, R3, N / (R1 * R2), true, ALONG>(s, P, pstride, estride, tw, tid, nthr); sync(); }
        if constexpr (PI::NST >= 2) { fft_stage<N, R2, N / R1, true, ALONG>(s, P, pstride, estride, tw, tid, nthr); sync(); }
        fft_stage<N, R1, N, true, ALONG>(s, P, pstride, estride, tw, tid, nthr);
    }
}

}  // namespace tddft
