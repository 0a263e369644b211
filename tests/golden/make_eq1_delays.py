"""Recompute tests/golden/eq1_delays.txt rows with exact rational arithmetic (no oracle, no
library): x = 4.15e6 * (f_c^-2 - f_top^-2) * DM / t_samp with f_c = f_top - c*df
(eq. 1).  Prints the rows; paste into eq1_delays.txt."""
from fractions import Fraction as F
import math

ROWS = [("150.0", "0.05", "0.1", 127, "3.0"), ("150.0", "0.05", "0.1", 64, "3.0"),
        ("150.0", "0.05", "0.1", 127, "6.3"), ("150.0", "0.05", "0.1", 1, "0.1"),
        ("150.0", "0.05", "0.1", 0, "6.3"),
        ("1582.0", "0.390625", "0.064", 1023, "2047.5"), ("1582.0", "0.390625", "0.064", 512, "1000.0"),
        ("143.0", "0.005859375", "0.0512", 1023, "102.35"),
        ("1500.0", "0.146484375", "0.064", 2047, "1535.5")]
for ft, df, ts, c, dm in ROWS:
    f_c = F(ft) - c * F(df)
    x = F(4150000) * (1 / f_c ** 2 - 1 / F(ft) ** 2) * F(dm) / F(ts)
    print(ft, df, ts, c, dm, "%.6f" % float(x), math.floor(x + F(1, 2)))
