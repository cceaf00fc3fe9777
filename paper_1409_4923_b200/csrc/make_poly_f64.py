"""Prints the polynomial coefficients of the fp64 kernels' own elementary functions (sim_f64.cuh: cos2pi_f64, log_u_f64,
sincospi_f64): interpolants at the Chebyshev nodes of the argument range, computed with mpmath at 60 digits and rounded
to double.  Run by hand when a range or degree changes; the output is pasted into sim_f64.cuh.  Not part of the oracle.
tests/test_poly_tables.py runs it and checks that the tables in sim_f64.cuh are its output."""
import mpmath as mp

mp.mp.dps = 60


def cheb_fit(f, a, b, n):
    xs = [(a + b) / 2 + (b - a) / 2 * mp.cos(mp.pi * (2 * k + 1) / (2 * n)) for k in range(n)]
    A, y = mp.matrix(n, n), mp.matrix(n, 1)
    for i, x in enumerate(xs):
        for j in range(n):
            A[i, j] = x ** j
        y[i] = f(x)
    c = mp.lu_solve(A, y)
    return [c[i] for i in range(n)]


def show(name, c):
    print(f"{name}[{len(c)}] = {{" + ", ".join(repr(float(v)) for v in c) + "};   // c0 + c1 z + ...")


sixteenth = mp.mpf(1) / 16
# force cosine cos2pi_f64: cos(2 pi r) as a degree-12 polynomial in u = r^2 on [0, 1/16], split into the two Horner chains
# in w = u^2 the kernel evaluates: E = (c12, c10, ..., c0), O = (c11, c9, ..., c1), highest coefficient first
c2 = cheb_fit(lambda z: mp.cos(2 * mp.pi * mp.sqrt(z)), mp.mpf(0), sixteenth, 13)
show("COS2PI_E", c2[12::-2])
show("COS2PI_O", c2[11::-2])
show("SINPI_C", cheb_fit(lambda z: mp.sin(mp.pi * mp.sqrt(z)) / mp.sqrt(z), mp.mpf(0), sixteenth, 8))   # sin(pi r) / r, z = r^2
show("COSPI_C", cheb_fit(lambda z: mp.cos(mp.pi * mp.sqrt(z)), mp.mpf(0), sixteenth, 8))                 # cos(pi r)
smax = (mp.sqrt(2) - 1) / (mp.sqrt(2) + 1)                     # s = f / (2 + f), f = m - 1, m in [sqrt(1/2), sqrt(2))
show("LOGP_C", cheb_fit(lambda z: (mp.log((1 + mp.sqrt(z)) / (1 - mp.sqrt(z))) / mp.sqrt(z) - 2) / z, mp.mpf(0), smax * smax * mp.mpf("1.0001"), 7))
ln2 = mp.log(2)
hi = mp.floor(ln2 * 2 ** 32) / 2 ** 32                           # 32 significant bits: k * LN2_HI is exact for |k| < 2^20
print("LN2_HI =", repr(float(hi)), " LN2_LO =", repr(float(ln2 - hi)))
# drive cosine of the inertial model (cos_drive_f64): sin(r) / r and cos(r) in z = r^2 on |r| <= pi/4, and pi/2 in three
# pieces (33 + 33 + 53 bits: k * PIO2_1 and k * PIO2_2 are exact for |k| < 2^20)
qz = (mp.pi / 4) ** 2 * mp.mpf("1.0001")
show("SIN_C", cheb_fit(lambda z: mp.sin(mp.sqrt(z)) / mp.sqrt(z), mp.mpf(0), qz, 8))
show("COS_C", cheb_fit(lambda z: mp.cos(mp.sqrt(z)), mp.mpf(0), qz, 8))
pio2 = mp.pi / 2
p1 = mp.floor(pio2 * 2 ** 32) / 2 ** 32
p2 = mp.floor((pio2 - p1) * 2 ** 65) / 2 ** 65
print("PIO2_1 =", repr(float(p1)), " PIO2_2 =", repr(float(p2)), " PIO2_3 =", repr(float(pio2 - p1 - p2)), " TWO_OVER_PI =", repr(float(2 / mp.pi)))
