"""Writes tests/golden/worked_example.txt from closed forms only (python `math`; no oracle, no CUDA).

The paper prints no worked numeric example for this path, so this fixture is a hand-derived one:
one group (G=2) of two labels sharing the support I = {0, 2} of d=3 features, chosen
so that every logit is ln 3, ln 4 or 0 and sigma / softplus are rationals / logs of integers:
  X = [[ln3, 9, 0], [0, -4, ln4]]   W = [[1, 0], [1, 1]]   idx = [[0, 2]]   y = [[1, 0], [0, 0]]   s = 1/B = 1/2
  z = [[ln3, ln3], [0, ln4]]                                        (z_l = <w_l, h_I>)
  loss = s * [ (ln4 - ln3) + ln4 + ln2 + ln5 ]                      (Eq. 3; softplus(ln n) = ln(n+1))
  dY = s * (sigma(z) - y) = [[-1/8, 3/8], [1/4, 2/5]]
  dW = dY^T H, H = X[:, I]  -> [[-ln3/8, ln4/4], [3 ln3/8, 2 ln4/5]]
  db = [1/8, 31/40]
  dX[:, I] += dY W           -> [[1/4, 0, 3/8], [13/20, 0, 2/5]]
Feature 1 (values 9, -4) is outside the support: a wrong gather index changes every number.
"""
import math
import os

ln = math.log
vals = {
    "X": [ln(3), 9.0, 0.0, 0.0, -4.0, ln(4)],
    "W": [1.0, 0.0, 1.0, 1.0],
    "idx": [0, 2],
    "rowptr": [0, 1, 1],
    "col": [0],
    "z": [ln(3), ln(3), 0.0, ln(4)],
    "loss": [0.5 * ((ln(4) - ln(3)) + ln(4) + ln(2) + ln(5))],
    "dY": [-1 / 8, 3 / 8, 1 / 4, 2 / 5],
    "dW": [-ln(3) / 8, ln(4) / 4, 3 * ln(3) / 8, 2 * ln(4) / 5],
    "db": [1 / 8, 31 / 40],
    "dX": [1 / 4, 0.0, 3 / 8, 13 / 20, 0.0, 2 / 5],
}
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "worked_example.txt")
with open(out, "w") as f:
    f.write("# hand-derived worked example (closed forms; see make_worked_example.py). B=2 d=3 L=2 G=2 K=2 s=0.5\n")
    f.write("# cites PAPER.md:72 (logit), :111 Eq.3 (BCE objective), :101 (dW), :103 (dX)\n")
    for k, v in vals.items():
        f.write(k + " " + " ".join(repr(x) for x in v) + "\n")
print(out)
