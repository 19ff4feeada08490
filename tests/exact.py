"""Exact-rational restatement of Eq. 4 used ONLY to pin the oracle.

Nothing here is shared with oracle/ or with the CUDA path: values are python Fractions / ints and
every IEEE rounding is done explicitly by `round_binary`, so a correctly rounded fp32 division or
multiplication has exactly one possible result and the oracle must reproduce it bit for bit.
Pure-python and slow: tiny shapes only.
"""
from fractions import Fraction


def round_binary(fr, p=24, emin=-126):
    """Round a Fraction to the nearest binary float with p significand bits (ties to even),
    gradual underflow below 2**emin.  p=24: binary32.  p=8: bfloat16.  No overflow handling."""
    fr = Fraction(fr)
    if fr == 0:
        return Fraction(0)
    s = -1 if fr < 0 else 1
    a = abs(fr)
    e = a.numerator.bit_length() - a.denominator.bit_length()
    if Fraction(2) ** e > a:
        e -= 1
    elif Fraction(2) ** (e + 1) <= a:
        e += 1
    assert Fraction(2) ** e <= a < Fraction(2) ** (e + 1)
    e = max(e, emin)
    ulp = Fraction(2) ** (e - (p - 1))
    n = round(a / ulp)          # python rounds Fractions half-to-even
    return s * n * ulp


def bf16_bits_to_fraction(b):
    b = int(b)
    sign = -1 if (b >> 15) & 1 else 1
    e = (b >> 7) & 0xFF
    m = b & 0x7F
    if e == 0:
        return sign * Fraction(m, 128) * Fraction(2) ** (-126)
    assert e != 255, "finite inputs only"
    return sign * (1 + Fraction(m, 128)) * Fraction(2) ** (e - 127)


def fraction_to_f32_bits(fr):
    """Bit pattern of a Fraction that is exactly representable in binary32."""
    fr = Fraction(fr)
    if fr == 0:
        return 0
    sign = 0x80000000 if fr < 0 else 0
    a = abs(fr)
    e = a.numerator.bit_length() - a.denominator.bit_length()
    if Fraction(2) ** e > a:
        e -= 1
    elif Fraction(2) ** (e + 1) <= a:
        e += 1
    if e < -126:
        m = a / Fraction(2) ** (-149)
        assert m.denominator == 1
        return sign | int(m)
    m = a / Fraction(2) ** (e - 23)
    assert m.denominator == 1 and (1 << 23) <= m < (1 << 24)
    return sign | ((e + 127) << 23) | (int(m) - (1 << 23))


def fraction_to_bf16_bits(fr):
    return fraction_to_f32_bits(fr) >> 16


F32_1E_5 = Fraction(0x27C5AC | 0x800000, 1 << 23) * Fraction(2) ** (0x6E - 127)   # 0x3727C5AC


def quant_row(x_bits):
    """Eq. 4 lines 1-2 for one row of bf16 bit patterns -> (a list[int], alpha Fraction(fp32 value))."""
    xs = [bf16_bits_to_fraction(b) for b in x_bits]
    amax = max([abs(v) for v in xs] + [Fraction(0)])
    alpha = round_binary(max(amax, F32_1E_5) / 127)            # fp32 division
    a = []
    for v in xs:
        t = round_binary(v / alpha)                            # fp32 division
        r = round(t)                                           # ties to even
        a.append(int(max(-127, min(127, r))))
    return a, alpha


def linear(x_bits_rows, w_rows, beta_f32):
    """Eq. 4 for tiny inputs.  x_bits_rows: [M][K] bf16 bits; w_rows: [N][K] ints in {-1,0,1};
    beta_f32: a Fraction that is an fp32 value.  Returns dict of python lists."""
    A, AL, ACC, Y32, YBF = [], [], [], [], []
    for xr in x_bits_rows:
        a, al = quant_row(xr)
        A.append(a)
        AL.append(al)
        s = round_binary(al * beta_f32)                        # fp32 multiply
        accs = [sum(ai * wi for ai, wi in zip(a, wr)) for wr in w_rows]
        ACC.append(accs)
        y = [round_binary(Fraction(c) * s) for c in accs]      # fp32 multiply ((float)acc is exact)
        Y32.append(y)
        YBF.append([round_binary(v, p=8) for v in y])
    return dict(a=A, alpha=AL, acc=ACC, y32=Y32, ybf16=YBF)
