"""Re-derive tests/golden/gubser_constants.txt from the printed formulas (Eq. 77, 116-120) with the
standard library only.  Calls neither oracle/ nor the CUDA library."""
import math

HBARC, C0, Q, TAU0 = 0.1973269804, 5.26, 1.0, 1.0
T0 = 0.4 / HBARC


def shape(tau, r):
    den = 1 + 2 * Q * Q * (tau * tau + r * r) + Q ** 4 * (tau * tau - r * r) ** 2
    return (2 * Q * tau) ** (2 / 3) / (tau * den ** (1 / 3))


def T(tau, r):
    return T0 * shape(tau, r) / shape(TAU0, 0.0)


def ur(tau, r):
    return 2 * Q * Q * r * tau / math.sqrt(1 + 2 * Q * Q * (tau * tau + r * r) + Q ** 4 * (tau * tau - r * r) ** 2)


if __name__ == "__main__":
    h = 0.3
    rows = [("T(1,0)", T(1, 0)), ("T(1,1)", T(1, 1)), ("T(1,2)", T(1, 2)), ("T(1,5)", T(1, 5)),
            ("ur(1,1)", ur(1, 1)), ("ur(1,2)", ur(1, 2)), ("s(T0)", 4 * C0 * T0 ** 3), ("e(T0)", 3 * C0 * T0 ** 4),
            ("sigma_2(h=0.3)", 10 / (7 * math.pi * h * h)), ("sigma_3(h=0.3)", 1 / (math.pi * h ** 3))]
    for k, v in rows:
        print(f"{k} {v:.9f}")
