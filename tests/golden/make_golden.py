"""Writes tests/golden/worked_example.txt.  Calls only oracle/brute.py (numpy
brute force); nothing from the CUDA path.  Run: python tests/golden/make_golden.py

The example is x = {0,1,2,3,4}, alpha = 2, c = 5 (hand-checkable):
  median 2; above-median residuals {1,2} -> sigma_upper = sqrt(2.5),
  s = 0.6745*sqrt(2.5); pass 1 by hand:
    5 s = 5.3323907
    u  = (x-2)/(5 s)       = {-0.37506630, -0.18753315, 0, 0.18753315, 0.37506630}
    ue = 2u for u<0        = {-0.75013260, -0.37506630, 0, 0.18753315, 0.37506630}
    w  = (1-ue^2)^2        = { 0.19123223,  0.73843992, 1, 0.93089947, 0.73843992}
    mu = sum(w x)/sum(w)   = 8.48489801 / 3.59901154 = 2.3575634
The remaining passes are written by the brute force below.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import brute  # noqa: E402


def main():
    x = [0.0, 1.0, 2.0, 3.0, 4.0]
    lines = ["# x = {0,1,2,3,4}, c = 5; written by tests/golden/make_golden.py from oracle/brute.py",
             "# key value"]
    mu, med, s, trace = brute.location(x, alpha=2.0, c=5.0, n_iter=5, history=True)
    lines.append("median %.17g" % med)
    lines.append("scale %.17g" % s)
    for k, m in enumerate(trace, 1):
        lines.append("alpha2_pass%d %.17g" % (k, m))
    mu1, _, _, trace1 = brute.location(x, alpha=1.0, c=5.0, n_iter=5, history=True)
    for k, m in enumerate(trace1, 1):
        lines.append("alpha1_pass%d %.17g" % (k, m))
    with open(os.path.join(HERE, "worked_example.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


if __name__ == "__main__":
    main()
