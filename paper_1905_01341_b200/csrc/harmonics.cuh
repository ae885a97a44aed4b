// Solid-harmonic machinery of the FMM ("multipole and local
// expansions ... truncated to the first p_fmm degrees (n = 0..p_fmm-1)").
// The paper defers every formula to its refs [30,32,33]; the
// convention used here is the one of DESIGN.md section 5:
//   R_l^m(r) = r^l P_l^m(cos th) e^{i m ph} / (l+m)!     (regular)
//   I_l^m(r) = (l-m)! P_l^m(cos th) e^{i m ph} / r^(l+1) (singular)
// with the Condon-Shortley phase, R_l^{-m} = (-1)^m conj R_l^m (same for I), so
// that 1/|x-y| = sum_{l,m} conj R_l^m(y-c) I_l^m(x-c).  Only m >= 0 is stored;
// a real field has C_l^{-m} = (-1)^m conj C_l^m, so an expansion is p^2 real
// numbers, laid out as  idx(l,0) = l^2,  idx(l,m,Re) = l^2+2m-1,  idx(l,m,Im) = l^2+2m.
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
BEM_HD int real_idx(int l, int m, int part) { return l * l + (m == 0 ? 0 : 2 * m - 1 + part); }

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

// decode a real-basis index c in [0, p^2) into (l, m, part)
BEM_HD void real_decode(int c, int *l, int *m, int *part)
{
    int ll = (int)sqrt((double)c);
    while (ll * ll > c) --ll;
    while ((ll + 1) * (ll + 1) <= c) ++ll;
    const int k = c - ll * ll;
    *l = ll;
    if (k == 0) { *m = 0; *part = 0; } else { *m = (k + 1) / 2; *part = (k + 1) & 1; }
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
BEM_HD double m2l_entry(const double *Ire, const double *Iim, int p, int cout, int cin)
{
    int l, m, po, j, k, pi;
    real_decode(cout, &l, &m, &po);
    real_decode(cin, &j, &k, &pi);
    const cplx Wp = tab_get(Ire, Iim, 2 * p - 1, j + l, k + m);
    const cplx Wm = tab_get(Ire, Iim, 2 * p - 1, j + l, -k + m);
    return real_entry(Wp, Wm, k, pi, po, (l & 1) ? -1.0 : 1.0);
}

// M2M:  Mt'_l^m = 2^-(l+1) sum_{j<=l,k} Mt_j^k conj R_{l-j}^{m-k}(that),
// that = (c_child - c_parent)/h_child.
BEM_HD double m2m_entry(const double *Rre, const double *Rim, int p, int cout, int cin)
{
    int l, m, po, j, k, pi;
    real_decode(cout, &l, &m, &po);
    real_decode(cin, &j, &k, &pi);
    if (j > l) return 0.0;
    cplx Wp = tab_get(Rre, Rim, p, l - j, m - k); Wp.im = -Wp.im;
    cplx Wm = tab_get(Rre, Rim, p, l - j, m + k); Wm.im = -Wm.im;
    return real_entry(Wp, Wm, k, pi, po, ldexp(1.0, -(l + 1)));
}

// L2L:  Lt'_j^k = sum_{l>=j,m} 2^-l Lt_l^m conj R_{l-j}^{m-k}(that),
// that = (c_child - c_parent)/h_child.  Output dof (j,k), input dof (l,m).
BEM_HD double l2l_entry(const double *Rre, const double *Rim, int p, int cout, int cin)
{
    int l, m, pi, j, k, po;
    real_decode(cout, &j, &k, &po);
    real_decode(cin, &l, &m, &pi);
    if (l < j) return 0.0;
    cplx Wp = tab_get(Rre, Rim, p, l - j, m - k); Wp.im = -Wp.im;
    cplx Wm = tab_get(Rre, Rim, p, l - j, -m - k); Wm.im = -Wm.im;
    return real_entry(Wp, Wm, m, pi, po, ldexp(1.0, -l));
}

}  // namespace bem
