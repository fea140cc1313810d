"""Regenerate the polynomial coefficients pasted into trig.cuh (run by hand; needs mpmath).

sin r = r + r u S(u), cos r = 1 - u/2 + u^2 C(u), u = r^2, |r| <= pi/4 (2 % margin):
S and C are degree-5 Chebyshev fits (near-minimax) of (sin r - r)/(r u) and (cos r - 1 + u/2)/u^2.
Approximation error with the coefficients rounded to fp64: 2^-55.2 (sin), 2^-59.4 (cos), relative.
"""
import mpmath as mp

mp.mp.dps = 60
U = (mp.pi / 4) ** 2 * mp.mpf("1.02")


def gs(u):
    if u == 0:
        return -mp.mpf(1) / 6
    r = mp.sqrt(u)
    return (mp.sin(r) - r) / (r * u)


def gc(u):
    if u == 0:
        return mp.mpf(1) / 24
    r = mp.sqrt(u)
    return (mp.cos(r) - 1 + u / 2) / (u * u)


if __name__ == "__main__":
    for name, g in (("kS", gs), ("kC", gc)):
        co = mp.chebyfit(g, [0, U], 6)          # highest degree first
        print(f"// {name}: highest degree first")
        print("    " + ", ".join(float(c).hex() for c in co))
    hi = float(mp.pi / 2)
    mid = float(mp.pi / 2 - hi)
    lo = float(mp.pi / 2 - hi - mid)
    print("// pi/2 split:", hi.hex(), mid.hex(), lo.hex())
    print("// 2/pi:", float(2 / mp.pi).hex())
