"""Writes gaussian_cvar.txt from scipy's normal distribution (closed form of PAPER.md (10)-(11) for N(0,1))."""
import os

from scipy.stats import norm

here = os.path.dirname(os.path.abspath(__file__))
with open(os.path.join(here, "gaussian_cvar.txt"), "w") as f:
    f.write("# alpha  CVaR_alpha(N(0,1)) = pdf(ppf(alpha))/(1-alpha)   [PAPER.md:97-101, eqs (10)-(11)]\n")
    for a in (0.5, 0.7, 0.9, 0.95, 0.99):
        f.write(f"{a} {norm.pdf(norm.ppf(a)) / (1 - a):.10f}\n")
