"""Writes chebyshev_T.txt from the defining three-term recurrence in exact integer arithmetic (no oracle, no CUDA)."""
import os

def main():
    T = [[1], [0, 1]]
    for n in range(1, 16):
        a = [0] + [2 * c for c in T[n]]
        b = T[n - 1] + [0] * (len(a) - len(T[n - 1]))
        T.append([x - y for x, y in zip(a, b)])
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "chebyshev_T.txt"), "w") as f:
        f.write("# degree : coefficients of T_degree(x), lowest power first (A&S Table 22.3)\n")
        for n in list(range(0, 9)) + [12, 16]:
            f.write(f"{n} : " + " ".join(str(c) for c in T[n]) + "\n")

if __name__ == "__main__":
    main()
