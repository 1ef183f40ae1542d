"""Writes the three literal values of tests/golden/paper_examples.json["counter_uniform"] with exact
Python integers (no numpy, nothing imported from this repo): the splitmix64 finaliser of
x = i + seed * 0x9E3779B97F4A7C15 (mod 2^64), then v = ((h >> 11) + 0.5) * (2 / 2^53) - 1 evaluated in IEEE
double arithmetic in that order (plain Python floats), as DESIGN.md reading 9 defines it.

    python tests/golden/make_counter_uniform.py        # prints the JSON fragment
"""
import json

M = (1 << 64) - 1


def h64(seed: int, i: int) -> int:
    x = (i + seed * 0x9E3779B97F4A7C15) & M
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & M
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & M
    return x ^ (x >> 31)


def value(seed: int, i: int) -> float:
    h = h64(seed, i)
    return (float(h >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0


if __name__ == "__main__":
    cases = [{"seed": s, "i": i, "h": h64(s, i), "v": value(s, i)} for s, i in [(7, 0), (12345, 1), (12346, 16777215)]]
    print(json.dumps(cases, indent=1))
