// su3.cuh — register-resident 3x3 complex algebra for the sweep kernels (sm_100a).
//
// A matrix is T v[18], element (i,j) at v[(i*3+j)*2 + c] (c = 0 re, 1 im): the same order in which
// the reals of a link sit in its 16-byte chunks in HBM, so chunk k of a link is
// v[k*NV .. k*NV+NV-1] and no shuffling is needed between load and use.  Every loop has compile-time
// bounds so that the arrays live in registers (the concern of PAPER.md:347).
#pragma once
#include <cuda_runtime.h>

namespace gf {

#define GF_DEV __device__ __forceinline__
#define RE(i, j) (((i) * 3 + (j)) * 2)
#define IM(i, j) (((i) * 3 + (j)) * 2 + 1)

template <class T>
struct Mat {
    T v[18];
};

template <class T>
GF_DEV void set_identity(Mat<T>& m) {
#pragma unroll
    for (int k = 0; k < 18; ++k) m.v[k] = T(0);
    m.v[RE(0, 0)] = T(1);
    m.v[RE(1, 1)] = T(1);
    m.v[RE(2, 2)] = T(1);
}
template <class T>
GF_DEV void set_zero(Mat<T>& m) {
#pragma unroll
    for (int k = 0; k < 18; ++k) m.v[k] = T(0);
}

// fused multiply-add in the matrix type (explicit: the compiler may contract a*b+c but not
// re-associate a*b - c*d + e, which would otherwise cost an extra rounding and instruction per term)
GF_DEV float fma_t(float a, float b, float c) { return __fmaf_rn(a, b, c); }
GF_DEV double fma_t(double a, double b, double c) { return __fma_rn(a, b, c); }

// third row from the first two: w = (u x v)^*
template <class T>
GF_DEV void reconstruct_row2(Mat<T>& m) {
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const int a = (j + 1) % 3, b = (j + 2) % 3;
        // (u_a v_b - u_b v_a), then conjugate
        T re = m.v[RE(0, a)] * m.v[RE(1, b)];
        re = fma_t(-m.v[IM(0, a)], m.v[IM(1, b)], re);
        re = fma_t(-m.v[RE(0, b)], m.v[RE(1, a)], re);
        re = fma_t(m.v[IM(0, b)], m.v[IM(1, a)], re);
        T im = m.v[RE(0, b)] * m.v[IM(1, a)];   // -Im(u_a v_b - u_b v_a)
        im = fma_t(m.v[IM(0, b)], m.v[RE(1, a)], im);
        im = fma_t(-m.v[RE(0, a)], m.v[IM(1, b)], im);
        im = fma_t(-m.v[IM(0, a)], m.v[RE(1, b)], im);
        m.v[RE(2, j)] = re;
        m.v[IM(2, j)] = im;
    }
}

// out(rows 0..NR-1) = G * M        (Step 2 for U_mu(x), with G = g3 g2 g1)
template <int NR, class T, class TG>
GF_DEV void mul_left(const Mat<TG>& G, const Mat<T>& M, Mat<T>& out) {
#pragma unroll
    for (int i = 0; i < NR; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = (T)G.v[RE(i, 0)] * M.v[RE(0, j)];
            T im = (T)G.v[RE(i, 0)] * M.v[IM(0, j)];
            re = fma_t(-(T)G.v[IM(i, 0)], M.v[IM(0, j)], re);
            im = fma_t((T)G.v[IM(i, 0)], M.v[RE(0, j)], im);
#pragma unroll
            for (int k = 1; k < 3; ++k) {
                const T gr = (T)G.v[RE(i, k)], gi = (T)G.v[IM(i, k)];
                re = fma_t(gr, M.v[RE(k, j)], re);
                re = fma_t(-gi, M.v[IM(k, j)], re);
                im = fma_t(gr, M.v[IM(k, j)], im);
                im = fma_t(gi, M.v[RE(k, j)], im);
            }
            out.v[RE(i, j)] = re;
            out.v[IM(i, j)] = im;
        }
}

// out(rows 0..NR-1) = M * G^dagger   (Step 2 for U_mu(x - mu)); needs rows 0..NR-1 of M only
template <int NR, class T, class TG>
GF_DEV void mul_right_dagger(const Mat<T>& M, const Mat<TG>& G, Mat<T>& out) {
#pragma unroll
    for (int i = 0; i < NR; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            // sum_k M_ik conj(G_jk)
            T re = M.v[RE(i, 0)] * (T)G.v[RE(j, 0)];
            T im = M.v[IM(i, 0)] * (T)G.v[RE(j, 0)];
            re = fma_t(M.v[IM(i, 0)], (T)G.v[IM(j, 0)], re);
            im = fma_t(-M.v[RE(i, 0)], (T)G.v[IM(j, 0)], im);
#pragma unroll
            for (int k = 1; k < 3; ++k) {
                const T gr = (T)G.v[RE(j, k)], gi = (T)G.v[IM(j, k)];
                re = fma_t(M.v[RE(i, k)], gr, re);
                re = fma_t(M.v[IM(i, k)], gi, re);
                im = fma_t(M.v[IM(i, k)], gr, im);
                im = fma_t(-M.v[RE(i, k)], gi, im);
            }
            out.v[RE(i, j)] = re;
            out.v[IM(i, j)] = im;
        }
}

// SU(2) element (g0,g1,g2,g3), Cayley-Klein form of Eq. (22):
//   [[g0 + i g3, g2 + i g1], [-g2 + i g1, g0 - i g3]] embedded in rows/cols (I,J).
// K <- g~ K : rows I and J of K are mixed.
template <int I, int J, class T>
GF_DEV void sub_left(Mat<T>& K, const T g[4]) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const T ar = K.v[RE(I, k)], ai = K.v[IM(I, k)], br = K.v[RE(J, k)], bi = K.v[IM(J, k)];
        // row I: (g0 + i g3) a + (g2 + i g1) b
        K.v[RE(I, k)] = g[0] * ar - g[3] * ai + g[2] * br - g[1] * bi;
        K.v[IM(I, k)] = g[0] * ai + g[3] * ar + g[2] * bi + g[1] * br;
        // row J: (-g2 + i g1) a + (g0 - i g3) b
        K.v[RE(J, k)] = -g[2] * ar - g[1] * ai + g[0] * br + g[3] * bi;
        K.v[IM(J, k)] = -g[2] * ai + g[1] * ar + g[0] * bi - g[3] * br;
    }
}
// K <- K g~^dagger : columns I and J of K are mixed.
template <int I, int J, class T>
GF_DEV void sub_right_dagger(Mat<T>& K, const T g[4]) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const T ar = K.v[RE(k, I)], ai = K.v[IM(k, I)], br = K.v[RE(k, J)], bi = K.v[IM(k, J)];
        // col I: a conj(g_II) + b conj(g_IJ) = a (g0 - i g3) + b (g2 - i g1)
        K.v[RE(k, I)] = ar * g[0] + ai * g[3] + br * g[2] + bi * g[1];
        K.v[IM(k, I)] = ai * g[0] - ar * g[3] + bi * g[2] - br * g[1];
        // col J: a conj(g_JI) + b conj(g_JJ) = a (-g2 - i g1) + b (g0 + i g3)
        K.v[RE(k, J)] = -ar * g[2] + ai * g[1] + br * g[0] - bi * g[3];
        K.v[IM(k, J)] = -ai * g[2] - ar * g[1] + bi * g[0] + br * g[3];
    }
}

// K += U          (Eq. (19), up-link term)
template <class A, class T>
GF_DEV void acc_plain(Mat<A>& K, const Mat<T>& U) {
#pragma unroll
    for (int k = 0; k < 18; ++k) K.v[k] += (A)U.v[k];
}
// K += W^dagger   (Eq. (19), down-link term)
template <class A, class T>
GF_DEV void acc_dagger(Mat<A>& K, const Mat<T>& W) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            K.v[RE(i, j)] += (A)W.v[RE(j, i)];
            K.v[IM(i, j)] -= (A)W.v[IM(j, i)];
        }
}

// MAG neighbourhood summary: Hermitian M_k = sum_up col_k col_k^dag + sum_down r r^dag,
// r = conj(row_k)^T, so that the local functional of Eq. (11) is sum_k (g M_k g^dag)_kk.
// Stored as its upper triangle: d = real diagonal, o = (0,1),(0,2),(1,2) complex.
template <class T>
struct Herm {
    T d[3];
    T o[6];
};
template <class T>
GF_DEV void set_zero(Herm<T>& h) {
#pragma unroll
    for (int k = 0; k < 3; ++k) h.d[k] = T(0);
#pragma unroll
    for (int k = 0; k < 6; ++k) h.o[k] = T(0);
}
template <class T>
GF_DEV void herm_expand(const Herm<T>& h, Mat<T>& m) {
#pragma unroll
    for (int k = 0; k < 3; ++k) { m.v[RE(k, k)] = h.d[k]; m.v[IM(k, k)] = T(0); }
    m.v[RE(0, 1)] = h.o[0]; m.v[IM(0, 1)] = h.o[1]; m.v[RE(1, 0)] = h.o[0]; m.v[IM(1, 0)] = -h.o[1];
    m.v[RE(0, 2)] = h.o[2]; m.v[IM(0, 2)] = h.o[3]; m.v[RE(2, 0)] = h.o[2]; m.v[IM(2, 0)] = -h.o[3];
    m.v[RE(1, 2)] = h.o[4]; m.v[IM(1, 2)] = h.o[5]; m.v[RE(2, 1)] = h.o[4]; m.v[IM(2, 1)] = -h.o[5];
}
template <class T>
GF_DEV void herm_compress(const Mat<T>& m, Herm<T>& h) {
#pragma unroll
    for (int k = 0; k < 3; ++k) h.d[k] = m.v[RE(k, k)];
    h.o[0] = m.v[RE(0, 1)]; h.o[1] = m.v[IM(0, 1)];
    h.o[2] = m.v[RE(0, 2)]; h.o[3] = m.v[IM(0, 2)];
    h.o[4] = m.v[RE(1, 2)]; h.o[5] = m.v[IM(1, 2)];
}
// M_k += col_k(U) col_k(U)^dagger : element (a,b) = U_ak conj(U_bk)
template <int KK, class A, class T>
GF_DEV void mag_acc_up(Herm<A>& Mk, const Mat<T>& U) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const A xr = (A)U.v[RE(a, KK)], xi = (A)U.v[IM(a, KK)];
        Mk.d[a] += xr * xr + xi * xi;
    }
    constexpr int PA[3] = {0, 0, 1}, PB[3] = {1, 2, 2};
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const A xr = (A)U.v[RE(PA[p], KK)], xi = (A)U.v[IM(PA[p], KK)];
        const A yr = (A)U.v[RE(PB[p], KK)], yi = (A)U.v[IM(PB[p], KK)];
        Mk.o[2 * p] += xr * yr + xi * yi;
        Mk.o[2 * p + 1] += xi * yr - xr * yi;
    }
}
// M_k += r r^dagger, r = conj(row_k(W))^T : element (a,b) = conj(W_ka) W_kb
template <int KK, class A, class T>
GF_DEV void mag_acc_down(Herm<A>& Mk, const Mat<T>& W) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const A xr = (A)W.v[RE(KK, a)], xi = (A)W.v[IM(KK, a)];
        Mk.d[a] += xr * xr + xi * xi;
    }
    constexpr int PA[3] = {0, 0, 1}, PB[3] = {1, 2, 2};
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const A xr = (A)W.v[RE(KK, PA[p])], xi = (A)W.v[IM(KK, PA[p])];
        const A yr = (A)W.v[RE(KK, PB[p])], yi = (A)W.v[IM(KK, PB[p])];
        Mk.o[2 * p] += xr * yr + xi * yi;
        Mk.o[2 * p + 1] += xr * yi - xi * yr;
    }
}

}  // namespace gf
