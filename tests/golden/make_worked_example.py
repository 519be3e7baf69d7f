"""Re-evaluates the hand enumeration of tests/golden/worked_example.txt with nothing but `math`.

Run:  python tests/golden/make_worked_example.py     (prints the key/value lines)
Each line below is one step of the hand derivation: the segment list is written out explicitly.
"""
import math

L = math.sqrt(1.0 + 0.375 ** 2)
kap = {(0, 0): 1.0, (0, 1): 0.5, (1, 0): 2.0, (1, 1): 0.25}
S = {(0, 0): 1.0, (0, 1): 0.25, (1, 0): 0.5, (1, 1): 2.0}
third = 1.0 / 3.0
rays = {
    "pm1": [((1, 0), 1.0 - third)],
    "p0": [((0, 0), 1.0), ((1, 0), third), ((1, 1), 1.0 - third)],
    "p1": [((0, 1), 1.0), ((1, 1), third)],
}
num = {c: 0.0 for c in kap}
den = {c: 0.0 for c in kap}
cnt = {c: 0 for c in kap}
exits = {}
for name, segs in rays.items():
    I = 0.0
    for cell, frac in segs:
        ds = frac * L
        dtau = kap[cell] * ds
        num[cell] += ds * I * (1.0 - math.exp(-dtau)) / dtau          # eq. 8, weighted by path length
        den[cell] += ds
        cnt[cell] += 1
        I = I * math.exp(-dtau) + S[cell] * (1.0 - math.exp(-dtau))   # eq. 7
    exits[name] = I
print("L", repr(L))
for c in sorted(kap):
    print("count_%d%d %d" % (c[0], c[1], cnt[c]))
print("total_segments", sum(cnt.values()))
print("sum_ds", repr(sum(den.values())))
for c in sorted(kap):
    print("Jin_%d%d %r" % (c[0], c[1], num[c] / den[c]))              # eqs. 11, 13 with N_d = 1
for k, v in exits.items():
    print("exit_%s %r" % (k, v))
