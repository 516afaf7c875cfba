// pm_ylm.h — real spherical harmonics Y_{lm}(u), m >= 0, of a unit vector u = (ux, 0, uz) in the xz-plane,
// Condon-Shortley phase, by the fully normalised three-term recurrence (host and device).
// The signed ux plays the role of sin(theta): azimuth pi gives (-1)^m automatically.  Y_{l,-m} = (-1)^m Y_{lm}.
//   Y_00 = 1/sqrt(4 pi);  Y_mm = ydiag[m] * ux * Y_{m-1,m-1},  ydiag[m] = -sqrt((2m+1)/(2m));
//   Y_lm = ya[lm] * (uz * Y_{l-1,m} - yb[lm] * Y_{l-2,m}),  ya = sqrt((4l^2-1)/(l^2-m^2)),
//   yb = sqrt(((l-1)^2-m^2)/(4(l-1)^2-1)).
// Used for the bipolar harmonics of eq. (22)'s angular part.
#pragma once

#if defined(__CUDACC__)
#define PM_HD __host__ __device__ __forceinline__
#else
#define PM_HD inline
#endif

namespace pm {

PM_HD int yidx(int l, int m) { return l * (l + 1) / 2 + m; }

PM_HD void ylm_fill(int lmax, double ux, double uz, const double* ya, const double* yb, const double* ydiag, double* Y)
{
    Y[0] = 0.28209479177387814347;
    for (int m = 0; m <= lmax; ++m) {
        if (m > 0) Y[yidx(m, m)] = ydiag[m] * ux * Y[yidx(m - 1, m - 1)];
        double p2 = 0.0, p1 = Y[yidx(m, m)];
        for (int l = m + 1; l <= lmax; ++l) {
            double cur = ya[yidx(l, m)] * (uz * p1 - yb[yidx(l, m)] * p2);
            Y[yidx(l, m)] = cur;
            p2 = p1; p1 = cur;
        }
    }
}

}  // namespace pm
