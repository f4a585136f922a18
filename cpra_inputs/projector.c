/*
 * cpra_inputs/projector.c -- forward model helper for the synthetic-input generator.
 *
 * Computes the line-integral projections P_n(z,u) = sum_s O(x(u,s), y(u,s), z) of a voxel
 * object rotated about the z axis (Eq. (2): the "3D to 2D real-space projection"
 * that defines a projected object).  Geometry:
 *     x = u cos(theta) - s sin(theta),   y = u sin(theta) + s cos(theta),
 * coordinates measured from the grid centre N/2, bilinear interpolation inside each z-slice,
 * zero outside the inner (unpadded) object grid.
 *
 * This is data generation only: it holds none of the CPRA iteration's arithmetic and is used
 * neither by oracle/ nor by the CUDA path -- only by cpra_inputs/generate.py.
 */
#include <math.h>
#include <stddef.h>

/* obj: [nin][nin][nin] (z,y,x), real part re and (optional, may be NULL) imaginary part im.
 * The inner grid sits centred in the N grid: inner index i <-> outer index i + (N-nin)/2.
 * out_re/out_im: [Np][N][N] as (n, z, u).  Rows z outside the inner grid are zero. */
void cpra_project(const double* re, const double* im, int nin, int N, int Np,
                  const double* angles, double* out_re, double* out_im)
{
    const int off = (N - nin) / 2;
    const double c = (double)(N / 2);            /* rotation centre, outer-grid index */
    /* the inner cube fits inside radius R about the centre in the (x,y) plane */
    const double R = 0.5 * nin * 1.4142135623730951 + 2.0;
    int u_lo = (int)floor(c - R), u_hi = (int)ceil(c + R);
    if (u_lo < 0) u_lo = 0;
    if (u_hi > N - 1) u_hi = N - 1;

    #pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int n = 0; n < Np; ++n) {
        for (int zi = 0; zi < nin; ++zi) {
            const double ct = cos(angles[n]), st = sin(angles[n]);
            const double* sl_re = re + (size_t)zi * nin * nin;
            const double* sl_im = im ? im + (size_t)zi * nin * nin : NULL;
            double* o_re = out_re + ((size_t)n * N + (zi + off)) * N;
            double* o_im = out_im ? out_im + ((size_t)n * N + (zi + off)) * N : NULL;
            for (int ui = u_lo; ui <= u_hi; ++ui) {
                const double u = ui - c;
                double acc_re = 0.0, acc_im = 0.0;
                for (int si = u_lo; si <= u_hi; ++si) {
                    const double s = si - c;
                    /* position in inner-grid index units */
                    const double x = u * ct - s * st + c - off;
                    const double y = u * st + s * ct + c - off;
                    const double fx = floor(x), fy = floor(y);
                    const int x0 = (int)fx, y0 = (int)fy;
                    if (x0 < -1 || y0 < -1 || x0 >= nin || y0 >= nin) continue;
                    const double wx = x - fx, wy = y - fy;
                    double v_re = 0.0, v_im = 0.0;
                    for (int dy = 0; dy < 2; ++dy) {
                        const int yy = y0 + dy;
                        if (yy < 0 || yy >= nin) continue;
                        const double wyy = dy ? wy : 1.0 - wy;
                        if (wyy == 0.0) continue;
                        for (int dx = 0; dx < 2; ++dx) {
                            const int xx = x0 + dx;
                            if (xx < 0 || xx >= nin) continue;
                            const double w = wyy * (dx ? wx : 1.0 - wx);
                            if (w == 0.0) continue;
                            v_re += w * sl_re[(size_t)yy * nin + xx];
                            if (sl_im) v_im += w * sl_im[(size_t)yy * nin + xx];
                        }
                    }
                    acc_re += v_re;
                    acc_im += v_im;
                }
                o_re[ui] = acc_re;
                if (o_im) o_im[ui] = acc_im;
            }
        }
    }
}
