"""Writes tests/golden/harmonic_trace.txt from a CLOSED FORM (no oracle, no CUDA).

Input family ("harmonic case"): q = 0 so every logit is 0 and every eligible token has
weight exp(0) = 1 (Eq. 1).  Block 1's value rows are all equal to
a * ones(d); every later block's value rows are 0.  With n tokens per block the App. A
recurrence gives A_t = n t and o^(t) = (a / t) ones(d), hence for a
probe of m coordinates (Eq. 2)

    d_scale^(1) = a sqrt(m)                       (x^(0) = 0, Alg. 1 l.1)
    d_scale^(t) = a sqrt(m) / (t (t - 1)),  t >= 2
    d_direction^(1) = 1  (zero-norm convention, reading R4)
    d_direction^(t) = 0, t >= 2                   (x^(t) parallel to x^(t-1))

and by Eq. 3 with strict '<' the first stable step is the smallest
t >= 2 with a sqrt(m) / (t (t-1)) < tau, and t* = that step + p - 1.
"""
import math
import os

A_VAL, M, TAU, P, T = 1.0, 32, 0.05, 5, 24

rows = []
for t in range(1, T + 1):
    ds = A_VAL * math.sqrt(M) if t == 1 else A_VAL * math.sqrt(M) / (t * (t - 1))
    dd = 1.0 if t == 1 else 0.0
    rows.append((t, ds, dd))
first = next(t for t, ds, dd in rows if t >= 2 and ds < TAU)
t_star = first + P - 1
here = os.path.dirname(os.path.abspath(__file__))
with open(os.path.join(here, "harmonic_trace.txt"), "w") as f:
    f.write("# closed form, see make_harmonic_golden.py; cites Eq. 1-3, App. A (PAPER.md:81,144,154,312)\n")
    f.write(f"# a={A_VAL} m={M} tau={TAU} p={P} T={T} first_stable={first} t_star={t_star}\n")
    f.write("# t d_scale d_direction\n")
    for t, ds, dd in rows:
        f.write(f"{t} {ds!r} {dd!r}\n")


# ---------------------------------------------------------------------------------------------------------------------
# Second closed form, with a NON-TRIVIAL direction term ("two-direction case"): q = 0 again (every weight is 1, A_t = n t).
# Block 1's value rows are all e_a, block 2's all e_b, every later block's all e_a again, with a != b two PROBE
# coordinates.  Then o^(t) = ((t - 1) e_a + e_b) / t for t >= 2 and o^(1) = e_a, so in the (e_a, e_b) plane
#     x^(t) = ((t - 1) / t, 1 / t),   x^(t) - x^(t-1) = (1, -1) / (t (t - 1))          (t >= 2)
#     d_scale^(t) = sqrt(2) / (t (t - 1)),   d_scale^(1) = 1
#     cos(x^(t), x^(t-1)) = ((t-1)(t-2) + 1) / sqrt(((t-1)^2 + 1) ((t-2)^2 + 1))   (integer vectors (t-1, 1), (t-2, 1))
#     d_direction^(2) = 1 - 1/sqrt(2),  d_direction^(1) = 1 (R4)
# A transposed operand, a dropped normalisation or a wrong sign in Eq. 2's cosine changes these values.
T2 = 12
with open(os.path.join(here, "two_direction_trace.txt"), "w") as f:
    f.write("# closed form, see make_harmonic_golden.py (second part); cites Eq. 1-2, App. A (PAPER.md:81,144,312)\n")
    f.write(f"# T={T2}\n")
    f.write("# t d_scale d_direction\n")
    for t in range(1, T2 + 1):
        if t == 1:
            ds, dd = 1.0, 1.0
        else:
            ds = math.sqrt(2.0) / (t * (t - 1))
            dd = 1.0 - ((t - 1) * (t - 2) + 1) / math.sqrt(((t - 1) ** 2 + 1) * ((t - 2) ** 2 + 1))
        f.write(f"{t} {ds!r} {dd!r}\n")
