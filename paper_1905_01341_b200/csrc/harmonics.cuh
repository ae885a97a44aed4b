// Solid-harmonic machinery of the FMM ("multipole and local
// expansions ... truncated to the first p_fmm degrees (n = 0..p_fmm-1)").
// The paper defers every formula to its refs [30,32,33]; the
// convention used here is the one of DESIGN.md section 5:
//   R_l^m(r) = r^l P_l^m(cos th) e^{i m ph} / (l+m)!     (regular)
//   I_l^m(r) = (l-m)! P_l^m(cos th) e^{i m ph} / r^(l+1) (singular)
// with the Condon-Shortley phase, R_l^{-m} = (-1)^m conj R_l^m (same for I), so
// that 1/|x-y| = sum_{l,m} conj R_l^m(y-c) I_l^m(x-c).  Only m >= 0 is stored;
// a real field has C_l^{-m} = (-1)^m conj C_l^m, so an expansion is p^2 real
// numbers.  Layout of a stored expansion (row of nst = 2 nre doubles): all REAL parts first,
// idx(l,m,Re) = l(l+1)/2 + m  (0 <= m <= l), padded to nre = a multiple of 8, then all
// IMAGINARY parts at the same place of the second half, idx(l,m,Im) = nre + l(l+1)/2 + m
// (the m = 0 slots stay zero), so that the two parts of a coefficient are exactly nre apart.
// The split is what makes the M2L matrices block diagonal:
// for an offset in the xz-plane every I_n^m(T) is real, so real parts map to real parts
// and imaginary parts to imaginary parts.  The layout is sized for pl >= p (the template
// bucket of the kernels); degrees p..pl-1 are kept zero.
//
// Box-scaled coefficients (h = box edge):  Mt_l^m = M_l^m / h^(l+1),
// Lt_l^m = L_l^m h^l.  With them every translation matrix depends only on the
// integer offset between boxes, not on the level.
#pragma once

#ifdef __CUDACC__
#define BEM_HD __host__ __device__ __forceinline__
#else
#define BEM_HD inline
#endif

namespace bem {

constexpr int P_MAX = 32;          // bem_setup rejects p > 32

BEM_HD int tri_idx(int l, int m) { return l * (l + 1) / 2 + m; }
BEM_HD int lay_nre(int pl) { return ((pl * (pl + 1) / 2 + 7) / 8) * 8; }
BEM_HD int lay_nst(int pl) { return 2 * lay_nre(pl); }
BEM_HD int real_idx(int l, int m, int part, int nre) { return part * nre + l * (l + 1) / 2 + m; }

// R_l^m(x,y,z) for 0 <= m <= l < p at tri_idx(l,m).
BEM_HD void eval_R(double x, double y, double z, int p, double *re, double *im)
{
    const double r2 = x * x + y * y + z * z;
    re[0] = 1.0; im[0] = 0.0;
    for (int m = 0; m < p; ++m) {
        const int mm = tri_idx(m, m);
        if (m > 0) {
            const int pm = tri_idx(m - 1, m - 1);
            const double f = -1.0 / (2.0 * m);           // R_m^m = -(x+iy)/(2m) R_{m-1}^{m-1}
            const double a = re[pm], b = im[pm];
            re[mm] = f * (x * a - y * b);
            im[mm] = f * (x * b + y * a);
        }
        for (int l = m + 1; l < p; ++l) {                // (l-m)(l+m) R_l^m = (2l-1) z R_{l-1}^m - r^2 R_{l-2}^m
            const int i0 = tri_idx(l, m), i1 = tri_idx(l - 1, m);
            const double inv = 1.0 / ((double)(l - m) * (double)(l + m));
            double vr = (2 * l - 1) * z * re[i1], vi = (2 * l - 1) * z * im[i1];
            if (l - 2 >= m) { const int i2 = tri_idx(l - 2, m); vr -= r2 * re[i2]; vi -= r2 * im[i2]; }
            re[i0] = vr * inv; im[i0] = vi * inv;
        }
    }
}

// I_l^m(x,y,z) for 0 <= m <= l < p at tri_idx(l,m);  (x,y,z) != 0.
BEM_HD void eval_I(double x, double y, double z, int p, double *re, double *im)
{
    const double r2 = x * x + y * y + z * z;
    const double ir2 = 1.0 / r2;
    re[0] = sqrt(ir2); im[0] = 0.0;
    for (int m = 0; m < p; ++m) {
        const int mm = tri_idx(m, m);
        if (m > 0) {
            const int pm = tri_idx(m - 1, m - 1);
            const double f = -(2.0 * m - 1.0) * ir2;     // I_m^m = -(2m-1)(x+iy)/r^2 I_{m-1}^{m-1}
            const double a = re[pm], b = im[pm];
            re[mm] = f * (x * a - y * b);
            im[mm] = f * (x * b + y * a);
        }
        for (int l = m + 1; l < p; ++l) {                // I_l^m = [(2l-1) z I_{l-1}^m - (l+m-1)(l-m-1) I_{l-2}^m]/r^2
            const int i0 = tri_idx(l, m), i1 = tri_idx(l - 1, m);
            double vr = (2 * l - 1) * z * re[i1], vi = (2 * l - 1) * z * im[i1];
            if (l - 2 >= m) {
                const int i2 = tri_idx(l - 2, m);
                const double c = (double)(l + m - 1) * (double)(l - m - 1);
                vr -= c * re[i2]; vi -= c * im[i2];
            }
            re[i0] = vr * ir2; im[i0] = vi * ir2;
        }
    }
}

struct cplx { double re, im; };

// value of a harmonic table at any (l, m), |m| <= l or zero outside
BEM_HD cplx tab_get(const double *re, const double *im, int lmax_excl, int l, int m)
{
    cplx v = {0.0, 0.0};
    if (l < 0 || l >= lmax_excl) return v;
    const int am = m < 0 ? -m : m;
    if (am > l) return v;
    const int i = tri_idx(l, am);
    v.re = re[i]; v.im = im[i];
    if (m < 0) { v.im = -v.im; if (am & 1) { v.re = -v.re; v.im = -v.im; } }
    return v;
}

// decode a stored index c in [0, nst) into (l, m, part); false for padding entries, degrees >= p and Im of m = 0
BEM_HD bool real_decode(int c, int p, int nre, int *l, int *m, int *part)
{
    const int im = c >= nre ? 1 : 0;
    const int t = im ? c - nre : c;
    int lt = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while (lt * (lt + 1) / 2 > t) --lt;
    while ((lt + 1) * (lt + 2) / 2 <= t) ++lt;
    *l = lt;
    *m = t - lt * (lt + 1) / 2;
    *part = im;
    return lt < p && !(im && *m == 0);
}

// One entry of a real translation matrix: the response at output dof
// (lo, mo, po) of the complex-linear map
//     out_{lo}^{mo} = scale * sum_k  in_{li}^{k} * W(lo, mo, li, k)
// to the unit real input dof (li, mi, pi), where the input obeys
// in^{-k} = (-1)^k conj in^k.  Wp = W(.., +mi), Wm = W(.., -mi).
BEM_HD double real_entry(cplx Wp, cplx Wm, int mi, int pi, int po, double scale)
{
    // u = 1 (pi=0) or i (pi=1);  val = u Wp + [mi>0] (-1)^mi conj(u) Wm
    double vr, vi;
    if (pi == 0) { vr = Wp.re; vi = Wp.im; } else { vr = -Wp.im; vi = Wp.re; }
    if (mi > 0) {
        const double s = (mi & 1) ? -1.0 : 1.0;
        if (pi == 0) { vr += s * Wm.re; vi += s * Wm.im; } else { vr += s * Wm.im; vi -= s * Wm.re; }
    }
    return scale * (po == 0 ? vr : vi);
}

// M2L:  Lt_l^m = (-1)^l sum_{j<p,k} Mt_j^k I_{j+l}^{k+m}(That),
// That = (c_target - c_source)/h.  Ire/Iim hold I up to degree 2p-2.
BEM_HD double m2l_entry(const double *Ire, const double *Iim, int p, int nre, int cout, int cin)
{
    int l, m, po, j, k, pi;
    if (!real_decode(cout, p, nre, &l, &m, &po) || !real_decode(cin, p, nre, &j, &k, &pi)) return 0.0;
    const cplx Wp = tab_get(Ire, Iim, 2 * p - 1, j + l, k + m);
    const cplx Wm = tab_get(Ire, Iim, 2 * p - 1, j + l, -k + m);
    return real_entry(Wp, Wm, k, pi, po, (l & 1) ? -1.0 : 1.0);
}

// M2M:  Mt'_l^m = 2^-(l+1) sum_{j<=l,k} Mt_j^k conj R_{l-j}^{m-k}(that),
// that = (c_child - c_parent)/h_child.
BEM_HD double m2m_entry(const double *Rre, const double *Rim, int p, int nre, int cout, int cin)
{
    int l, m, po, j, k, pi;
    if (!real_decode(cout, p, nre, &l, &m, &po) || !real_decode(cin, p, nre, &j, &k, &pi)) return 0.0;
    if (j > l) return 0.0;
    cplx Wp = tab_get(Rre, Rim, p, l - j, m - k); Wp.im = -Wp.im;
    cplx Wm = tab_get(Rre, Rim, p, l - j, m + k); Wm.im = -Wm.im;
    return real_entry(Wp, Wm, k, pi, po, ldexp(1.0, -(l + 1)));
}

// L2L:  Lt'_j^k = sum_{l>=j,m} 2^-l Lt_l^m conj R_{l-j}^{m-k}(that),
// that = (c_child - c_parent)/h_child.  Output dof (j,k), input dof (l,m).
BEM_HD double l2l_entry(const double *Rre, const double *Rim, int p, int nre, int cout, int cin)
{
    int l, m, pi, j, k, po;
    if (!real_decode(cout, p, nre, &j, &k, &po) || !real_decode(cin, p, nre, &l, &m, &pi)) return 0.0;
    if (l < j) return 0.0;
    cplx Wp = tab_get(Rre, Rim, p, l - j, m - k); Wp.im = -Wp.im;
    cplx Wm = tab_get(Rre, Rim, p, l - j, -m - k); Wm.im = -Wm.im;
    return real_entry(Wp, Wm, m, pi, po, ldexp(1.0, -l));
}

}  // namespace bem
