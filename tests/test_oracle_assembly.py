"""Pins for the oracle's Fourier-slice assembly (P:35-44 Fourier slice theorem; P:72 Step D).

The paper only says "interpolate": the scheme (polar bilinear gather, reading A17) is this build's.  Every step of it is
pinned: the discrete Fourier-slice identity at theta = 0 and 90 degrees (exact), Hermitian symmetry for a real object, the
centring convention, an analytic Gaussian for general angles (geometry, with sign / swap controls), the averaging of
duplicate rays, and the interpolation weights themselves (exact on a spectrum that is bilinear in angle and radius).  How
close the scheme comes to the continuous transform is a property of the method: measured (the Gaussian case), not pinned."""
import numpy as np

import cpra_inputs
from oracle import Oracle, fft2


def _padded(obj, N):
    nin = obj.shape[0]
    off = (N - nin) // 2
    v = np.zeros((N, N, N), dtype=obj.dtype)
    v[off:off + nin, off:off + nin, off:off + nin] = obj
    return v


def test_fourier_slice_identity_discrete(tiny_problem):
    # F2[sum_y O](kz, kx) == F3[O](kz, 0, kx)  (theta = 0), and the theta = 90 degree analogue:
    # P(z,u) = sum_s O[z][y=u][x=-s]  =>  F2[P](kz, ku) == F3[O](kz, ky=ku, kx=0)
    p = tiny_problem
    N = p.N
    F3 = np.fft.fftn(_padded(p.obj, N))
    F2_0 = fft2(p.projections[0])
    assert np.abs(F2_0 - F3[:, 0, :]).max() < 1e-9 * np.abs(F3).max()
    n90 = p.Np // 2
    assert abs(p.angles[n90] - np.pi / 2) < 1e-15
    F2_90 = fft2(p.projections[n90])
    assert np.abs(F2_90 - F3[:, :, 0]).max() < 1e-9 * np.abs(F3).max()


def _assemble_true(p):
    o = Oracle(p.N, p.Np)
    o.set_data(np.ones((p.Np, p.N, p.N)), None, p.angles)
    o.set_support(np.ones((p.Np, p.N, p.N), np.uint8))
    o.set_estimate(p.projections)
    return o.assemble_3d()


def test_assembly_exact_on_the_measured_planes(tiny_problem):
    p = tiny_problem
    N, h = p.N, p.N // 2
    vol, w = _assemble_true(p)
    F3 = np.fft.fftn(_padded(p.obj, N))
    k = np.fft.fftfreq(N, 1.0 / N).astype(int)
    inside = np.abs(k) <= h - 1
    scale = np.abs(F3).max()
    # plane ky = 0 (theta = 0 slice) and plane kx = 0 (theta = 90 degrees slice); the axis rho = 0
    # is by definition the mean over ALL slices (bilinear rotation does not conserve mass exactly)
    off_axis = inside & (k != 0)
    assert np.abs(vol[:, 0, :][:, off_axis] - F3[:, 0, :][:, off_axis]).max() < 1e-9 * scale
    assert np.abs(vol[:, :, 0][:, off_axis] - F3[:, :, 0][:, off_axis]).max() < 1e-9 * scale
    dc = np.mean([np.fft.fft(pr[:, :].sum(axis=1)) for pr in p.projections], axis=0)   # F2[P_n](kz, 0)
    assert np.abs(vol[:, 0, 0] - dc).max() < 1e-9 * scale
    assert np.abs(vol[:, 0, 0] - F3[:, 0, 0]).max() < 2e-3 * scale
    # weights: 1 inside the measured cylinder rho <= N/2 - 1, 0 outside, and 0 value outside
    KY, KX = np.meshgrid(k, k, indexing="ij")
    rho = np.sqrt(KY ** 2 + KX ** 2)
    assert np.array_equal(w[3] == 1.0, rho <= h - 1)
    assert np.abs(vol[:, rho > h - 1]).max() == 0.0


def test_assembly_hermitian_for_real_object(tiny_problem):
    p = tiny_problem
    vol, w = _assemble_true(p)
    N = p.N
    idx = (-np.arange(N)) % N
    mirrored = np.conj(vol[idx][:, idx][:, :, idx])
    # exclude the Nyquist planes, which are their own mirror only up to the sampled half
    k = np.fft.fftfreq(N, 1.0 / N).astype(int)
    ok = np.abs(k) < N // 2
    sub = np.ix_(ok, ok, ok)
    assert np.abs(vol[sub] - mirrored[sub]).max() < 1e-9 * np.abs(vol).max()


def _gaussian_case(Np, N=32, sig=1.6, r0=(2.0, -1.0, 1.5), wrong=None):
    """Analytic off-centre Gaussian blob at (x0,y0,z0) from the grid centre: its projection along
    any direction is again a Gaussian, centred at u0 = x0 cos(th) + y0 sin(th) (from
    x = u cos - s sin, y = u sin + s cos), so the slices are exact up to aliasing (~1e-6)."""
    x0, y0, z0 = r0
    c = N // 2
    g = np.arange(N) - c
    obj = np.exp(-0.5 * (((g - z0) / sig) ** 2)[:, None, None] - 0.5 * (((g - y0) / sig) ** 2)[None, :, None]
                 - 0.5 * (((g - x0) / sig) ** 2)[None, None, :])
    F3 = np.fft.fftn(obj)
    angles = np.pi * np.arange(Np) / Np
    P = np.empty((Np, N, N), complex)
    for n, th in enumerate(angles):
        u0 = x0 * np.cos(th) + y0 * np.sin(th)
        if wrong == "swap":
            u0 = x0 * np.sin(th) + y0 * np.cos(th)
        if wrong == "sign":
            u0 = x0 * np.cos(th) - y0 * np.sin(th)
        P[n] = np.sqrt(2 * np.pi) * sig * np.exp(-0.5 * (((g - z0) / sig) ** 2)[:, None]
                                                 - 0.5 * (((g - u0) / sig) ** 2)[None, :])
    o = Oracle(N, Np)
    o.set_data(np.ones((Np, N, N)), None, angles)
    o.set_support(np.ones((Np, N, N), np.uint8))
    o.set_estimate(P)
    vol, w = o.assemble_3d()
    k = np.fft.fftfreq(N, 1.0 / N).astype(int)
    low = np.abs(k) <= 8
    sub = np.ix_(low, low, low)
    return np.linalg.norm((vol[sub] - F3[sub]).ravel()) / np.linalg.norm(F3[sub].ravel())


def test_assembly_geometry_against_analytic_gaussian():
    e16, e64 = _gaussian_case(16), _gaussian_case(64)
    assert e64 < 0.02, e64                       # only interpolation error is left
    assert e64 < e16                             # and it shrinks with the number of slices
    # a swapped sin/cos or a flipped rotation sense in the slice placement would show as O(1)
    assert _gaussian_case(64, wrong="swap") > 10 * e64
    assert _gaussian_case(64, wrong="sign") > 10 * e64


def test_assembly_merges_duplicate_rays_on_a_360_scan():
    # over [0, 360) the direction of slice n's negative ray equals slice n+Np/2's positive ray:
    # duplicates are averaged, so a consistent data set gives the same volume as the 180 degree scan
    N, nin = 16, 8
    rng = np.random.default_rng(3)
    obj = rng.uniform(size=(nin, nin, nin))
    a180 = np.pi * np.arange(4) / 4
    a360 = 2 * np.pi * np.arange(8) / 8
    vols = []
    for ang in (a180, a360):
        P = cpra_inputs.project(obj, N, ang)
        o = Oracle(N, len(ang))
        o.set_data(np.ones((len(ang), N, N)), None, ang)
        o.set_support(np.ones((len(ang), N, N), np.uint8))
        o.set_estimate(P)
        vols.append(o.assemble_3d()[0])
    F3 = np.fft.fftn(_padded(obj, N))
    # on the exactly measured plane ky = 0 both agree with the truth
    k = np.fft.fftfreq(N, 1.0 / N).astype(int)
    inside = np.abs(k) <= N // 2 - 1
    off_axis = inside & (k != 0)
    for v in vols:
        assert np.abs(v[:, 0, :][:, off_axis] - F3[:, 0, :][:, off_axis]).max() < 1e-9 * np.abs(F3).max()


def test_assembly_averages_duplicate_rays_carrying_different_data():
    """Step (ii) of the assembly: on a [0, 360) scan the ku <= 0 half of slice n points the same way
    as the ku >= 0 half of slice n + Np/2; the two are ONE ray whose samples are the MEAN of the
    contributors.  Give every slice a different constant spectrum c_n (g_n = c_n delta at the centre
    pixel: F2 = c_n (-1)^(kz+ku), which step (i) turns into the constant c_n): the voxels on the
    ray of direction theta_n then hold (c_n + c_{n+Np/2}) / 2 -- not c_n, not c_{n+Np/2} (first / last
    contributor wins) -- and the axis rho = 0 holds the mean of all c_n."""
    N, Np, h = 16, 4, 8
    c = np.array([1.0 + 0.5j, -2.0 + 1.0j, 4.0 - 1.5j, 0.5 + 3.0j])
    ang = 2 * np.pi * np.arange(Np) / Np                     # 0, 90, 180, 270 degrees
    P = np.zeros((Np, N, N), complex)
    P[:, h, h] = c
    o = Oracle(N, Np)
    o.set_data(np.ones((Np, N, N)), None, ang)
    o.set_support(np.ones((Np, N, N), np.uint8))
    o.set_estimate(P)
    vol, w = o.assemble_3d()
    m02, m13 = (c[0] + c[2]) / 2, (c[1] + c[3]) / 2
    for kz in (0, 1, 5, -3):
        for r in range(1, h):
            sg = (-1.0) ** (kz + r)                          # step (iv): (-1)^(kx+ky+kz)
            assert abs(vol[kz % N, 0, r] - sg * m02) < 1e-13, (kz, r)          # direction 0: slices 0 (+) and 2 (-)
            assert abs(vol[kz % N, 0, -r] - sg * m02) < 1e-13, (kz, r)         # direction 180
            assert abs(vol[kz % N, r, 0] - sg * m13) < 1e-13, (kz, r)          # direction 90: slices 1 (+) and 3 (-)
            assert abs(vol[kz % N, -r, 0] - sg * m13) < 1e-13, (kz, r)         # direction 270
        assert abs(vol[kz % N, 0, 0] - (-1.0) ** kz * c.mean()) < 1e-13
    # on the diagonal (45 degrees: halfway between two merged rays; rho = r sqrt(2) is bracketed by
    # constant radial samples) the bilinear value is the mean of the two ray means
    assert abs(vol[0, 2, 2] - (m02 + m13) / 2) < 1e-13
    assert abs(m02 - c[0]) > 0.5 and abs(m02 - c[2]) > 0.5   # averaging is distinguishable from one winner


def test_assembly_interpolation_is_exact_on_a_field_bilinear_in_angle_and_radius():
    """Step (iii) of the assembly interpolates bilinearly in (phi, rho) between the two rays that bracket a voxel and
    the radial samples floor(rho), floor(rho) + 1: it must reproduce f = a + rho (b phi + c) + d kz exactly wherever the
    bracket does not straddle the 0 / 2 pi cut.  Swapped or mis-normalised weights, a wrong bracketing ray, an off-by-one
    radial sample or a lost sign factor all fail."""
    N, Np = 32, 12
    a, b, c, d = 0.7, 0.31, -0.45, 0.05
    ang = np.pi * np.arange(Np) / Np
    k = np.fft.fftfreq(N, 1.0 / N).astype(int)                      # signed frequency of native index i
    KZ, KU = np.meshgrid(k, k, indexing="ij")
    G = np.empty((Np, N, N), complex)
    for n, th in enumerate(ang):
        phi = np.where(KU >= 0, th, th + np.pi)                       # the ray a sample belongs to
        C = a + np.abs(KU) * (b * phi + c) + d * KZ + 1j * (0.2 + 0.1 * np.abs(KU) * phi)      # centred spectrum wanted
        E = C * (-1.0) ** ((KZ + KU) % 2)                             # step (i) multiplies by (-1)^(kz + ku)
        G[n] = np.fft.ifft2(E)
    o = Oracle(N, Np)
    o.set_data(np.ones((Np, N, N)), None, ang)
    o.set_support(np.ones((Np, N, N), np.uint8))
    o.set_estimate(G)
    vol, w = o.assemble_3d()
    Z, Y, X = np.meshgrid(k, k, k, indexing="ij")
    rho = np.hypot(X, Y)
    phi = np.mod(np.arctan2(Y, X), 2 * np.pi)
    want = (a + rho * (b * phi + c) + d * Z + 1j * (0.2 + 0.1 * rho * phi)) * (-1.0) ** ((X + Y + Z) % 2)
    last = ang[-1] + np.pi                                            # the last ray before the cut
    ok = (rho > 0) & (rho <= N // 2 - 1) & (phi <= last)
    assert ok.mean() > 0.6
    assert np.abs(vol[ok] - want[ok]).max() < 1e-11
    assert np.all(w[ok] == 1.0) and np.all(w[rho > N // 2 - 1] == 0.0) and np.all(vol[rho > N // 2 - 1] == 0.0)
    # on the axis rho = 0 the mean of the slices' DC samples: a + d kz (+ 0.2 i)
    axis = (X == 0) & (Y == 0)
    assert np.abs(vol[axis] - want[axis]).max() < 1e-12
