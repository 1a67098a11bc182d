"""Generates the polynomial coefficients pasted into ms_math.cuh (run by hand; not used at build time).

  log core : ln(m) = 2 s + s^3 * PL(s^2),  s = f/(2+f), m = 1+f in [sqrt(1/2), sqrt(2)]
             PL(z) ~ (2 atanh(sqrt z) - 2 sqrt z) / z^(3/2)            on z in [0, (3-2 sqrt 2)^2]
  exp core : expm1(r) = r + r^2 * PE(r),  |r| <= ln(2)/2
             PE(r) ~ (e^r - 1 - r) / r^2
  sincospi : sin(pi r) = r * PS(r^2), cos(pi r) = 1 + r^2 * PC(r^2),  |r| <= 1/4

Near-minimax fits by Chebyshev interpolation in 60-digit arithmetic (mpmath.chebyfit); the script prints
each coefficient as a C hex-float and the measured maximum error of the fitted form.
"""
import mpmath as mp

mp.mp.dps = 60


def hexf(x):
    return float(x).hex()


def show(name, coeffs):
    print(f"// {name}: highest degree first")
    for c in coeffs:
        print(f"    {hexf(c)},  // {mp.nstr(c, 20)}")


def fit(f, a, b, n):
    return mp.chebyfit(f, [a, b], n)


def main():
    # ---- log
    smax = 3 - 2 * mp.sqrt(2)
    zmax = smax ** 2 * mp.mpf("1.02")

    def gl(z):
        if z < mp.mpf(10) ** -30:
            return mp.mpf(2) / 3
        s = mp.sqrt(z)
        return (2 * mp.atanh(s) - 2 * s) / (s ** 3)

    pl = fit(gl, 0, zmax, 8)
    show("PL", pl)
    worst = 0
    for i in range(1, 2000):
        s = smax * i / 2000
        approx = 2 * s + s ** 3 * mp.polyval([mp.mpf(float(c)) for c in pl], s * s)
        worst = max(worst, abs(approx / (2 * mp.atanh(s)) - 1))
    print("// log core max rel err", mp.nstr(worst, 5))

    # ---- expm1
    rmax = mp.log(2) / 2 * mp.mpf("1.01")

    def ge(r):
        if abs(r) < mp.mpf(10) ** -25:
            return mp.mpf(1) / 2 + r / 6
        return (mp.expm1(r) - r) / (r * r)

    pe = fit(ge, -rmax, rmax, 10)
    show("PE", pe)
    worst = 0
    for i in range(-2000, 2001):
        if i == 0:
            continue
        r = rmax * i / 2000
        approx = r + r * r * mp.polyval([mp.mpf(float(c)) for c in pe], r)
        worst = max(worst, abs(approx / mp.expm1(r) - 1))
    print("// expm1 core max rel err", mp.nstr(worst, 5))

    # ---- sinpi / cospi on |r| <= 1/4
    zq = mp.mpf(1) / 16 * mp.mpf("1.02")

    def gs(z):
        if z < mp.mpf(10) ** -30:
            return mp.pi
        r = mp.sqrt(z)
        return mp.sin(mp.pi * r) / r

    def gc(z):
        if z < mp.mpf(10) ** -30:
            return -mp.pi ** 2 / 2
        r = mp.sqrt(z)
        return (mp.cos(mp.pi * r) - 1) / z

    ps = fit(gs, 0, zq, 7)
    pc = fit(gc, 0, zq, 7)
    show("PS", ps)
    show("PC", pc)
    ws = wc = 0
    for i in range(1, 2001):
        r = mp.mpf(i) / 8000
        a = r * mp.polyval([mp.mpf(float(c)) for c in ps], r * r)
        b = 1 + r * r * mp.polyval([mp.mpf(float(c)) for c in pc], r * r)
        ws = max(ws, abs(a / mp.sin(mp.pi * r) - 1))
        wc = max(wc, abs(b / mp.cos(mp.pi * r) - 1))
    print("// sinpi / cospi core max rel err", mp.nstr(ws, 5), mp.nstr(wc, 5))


if __name__ == "__main__":
    main()


def atan_turns():
    """atan(t) / (2 pi) = t * PA(t^2) on |t| <= sqrt(2) - 1 (the FastRambo inverse's azimuth, in turns)."""
    zmax = (mp.sqrt(2) - 1) ** 2 * mp.mpf("1.01")

    def g(z):
        if z < mp.mpf(10) ** -30:
            return 1 / (2 * mp.pi)
        t = mp.sqrt(z)
        return mp.atan(t) / (2 * mp.pi * t)

    pa = fit(g, 0, zmax, 11)
    show("PA", pa)
    worst = 0
    for i in range(1, 3001):
        t = (mp.sqrt(2) - 1) * i / 3000
        ap = t * mp.polyval([mp.mpf(float(c)) for c in pa], t * t)
        worst = max(worst, abs(ap / (mp.atan(t) / (2 * mp.pi)) - 1))
    print("// atan (turns) core max rel err", mp.nstr(worst, 5))


if __name__ == "__main__":
    atan_turns()
