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
