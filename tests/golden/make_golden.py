"""Writes the small text fixtures under tests/golden/.  Run: python tests/golden/make_golden.py

Every stored value comes from a closed form evaluated here with the Python standard library (math.erf,
math.sin ...) -- nothing is produced by the CUDA path, and nothing by the oracle either: the fixtures
are what the ORACLE is checked against (tests/test_golden.py).  The paper prints no worked numeric
example (its results are figures), so the closed forms below are the values "the mathematics fixes":

  green_gauss2.txt   G(r) = -erf(r / (sqrt(2) eps)) / (4 pi r), G(0) = -1 / ((2 pi)^(3/2) eps)
                     (2nd-order Gaussian-regularised kernel; reading A10)
  gaussian_blob.txt  potential of one Gaussian charge (strength q, width sigma) convolved with G_eps:
                     phi(r) = -q erf(r / (sqrt(2) s)) / (4 pi r), s^2 = sigma^2 + eps^2  (pin P5)
  fd2_dirichlet.txt  amplification A = pi^2 sum m_a^2 / ((4/h^2) sum sin^2(m_a pi h / 2)) of the product
                     of sines under the 7-point stencil (Table 1 row 1; pin P3)
  green_orders.txt   the regularised kernels at the origin and far away, where closed forms need no special
                     function: 3-D G_P(0) = -(1, 3/2, 15/8, 35/16, 315/128) / ((2 pi)^(3/2) eps) for P = 2 .. 10,
                     spectrally compact G(0) = -1 / (2 pi h); 2-D G_P(0) = (ln(2 eps^2) - gamma) / (4 pi)
                     - (1 / 4 pi) sum_{n < P/2} 1/n; far field -1 / (4 pi r) and ln(r) / (2 pi)
                     (readings A25, A26, A28)
  periodic_mode.txt  phi = -(a cos th + b sin th) / (4 pi^2 (p^2 + q^2)) for one Fourier mode (eq. 5,
                     PAPER.md:50; pin P2) at a few cell-centre points of the 64^2 grid of cfg 1
"""
import math
from pathlib import Path

HERE = Path(__file__).resolve().parent


def main():
    with open(HERE / "green_gauss2.txt", "w") as f:
        f.write("# r eps G(r)   -- PAPER.md:189, DESIGN.md A10\n")
        for eps in (0.0078125, 0.05):
            for r in (0.0, 0.25 * eps, eps, 3.0 * eps, 0.5, 1.7320508075688772):
                g = -1.0 / ((2 * math.pi) ** 1.5 * eps) if r == 0.0 else -math.erf(r / (math.sqrt(2) * eps)) / (4 * math.pi * r)
                f.write(f"{r!r} {eps!r} {g!r}\n")
    with open(HERE / "gaussian_blob.txt", "w") as f:
        f.write("# n sigma_over_h eps_over_h q ix iy iz phi   -- blob centred at cell centre (n/2,n/2,n/2)+0.5, h=1/n; pin P5\n")
        n, q = 64, 1.25
        h = 1.0 / n
        for sh, eh in ((2.0, 2.0), (2.0, 1.5)):
            s = math.sqrt((sh * h) ** 2 + (eh * h) ** 2)
            for (ix, iy, iz) in ((32, 32, 32), (33, 32, 32), (40, 20, 36), (5, 60, 11)):
                r = h * math.sqrt((ix - 32) ** 2 + (iy - 32) ** 2 + (iz - 32) ** 2)
                phi = -q / ((2 * math.pi) ** 1.5 * s) if r == 0 else -q * math.erf(r / (math.sqrt(2) * s)) / (4 * math.pi * r)
                f.write(f"{n} {sh!r} {eh!r} {q!r} {ix} {iy} {iz} {phi!r}\n")
    with open(HERE / "fd2_dirichlet.txt", "w") as f:
        f.write("# nc mx my mz A   -- psi = A prod sin(m_a pi x_a) solves the 7-point system for f = -pi^2 sum m^2 prod sin; PAPER.md:162\n")
        for nc, m in ((16, (1, 2, 3)), (32, (3, 5, 2)), (64, (7, 1, 4))):
            h = 1.0 / nc
            lam = sum(-(4 / h ** 2) * math.sin(mm * math.pi * h / 2) ** 2 for mm in m)
            A = -(math.pi ** 2) * sum(mm * mm for mm in m) / lam
            f.write(f"{nc} {m[0]} {m[1]} {m[2]} {A!r}\n")
    with open(HERE / "green_orders.txt", "w") as f:
        f.write("# dim order r eps G   -- order 0 = spectrally compact kernel (eps = h); PAPER.md:189, DESIGN.md A25 / A26 / A28\n")
        gamma = 0.5772156649015329
        c3 = {2: 1.0, 4: 1.5, 6: 15.0 / 8, 8: 35.0 / 16, 10: 315.0 / 128}
        for eps in (0.0078125, 0.05):
            for order in (2, 4, 6, 8, 10):
                f.write(f"3 {order} 0.0 {eps!r} {-c3[order] / ((2 * math.pi) ** 1.5 * eps)!r}\n")
                f.write(f"3 {order} {40 * eps!r} {eps!r} {-1.0 / (4 * math.pi * 40 * eps)!r}\n")
                g0 = (math.log(2 * eps * eps) - gamma) / (4 * math.pi) - sum(1.0 / n for n in range(1, order // 2)) / (4 * math.pi)
                f.write(f"2 {order} 0.0 {eps!r} {g0!r}\n")
                f.write(f"2 {order} {40 * eps!r} {eps!r} {math.log(40 * eps) / (2 * math.pi)!r}\n")
            f.write(f"3 0 0.0 {eps!r} {-1.0 / (2 * math.pi * eps)!r}\n")
    with open(HERE / "periodic_mode.txt", "w") as f:
        f.write("# n p q a b ix iy phi dphidx dphidy   -- f = a cos th + b sin th, th = 2 pi (p x + q y), x=(ix+.5)/n; PAPER.md:50, :141\n")
        n = 64
        for (p, q, a, b) in ((3, 5, 0.7, -1.1), (8, 1, -0.3, 0.9)):
            for (ix, iy) in ((0, 0), (17, 42), (63, 5)):
                x, y = (ix + 0.5) / n, (iy + 0.5) / n
                th = 2 * math.pi * (p * x + q * y)
                k2 = 4 * math.pi ** 2 * (p * p + q * q)
                phi = -(a * math.cos(th) + b * math.sin(th)) / k2
                dth = -(-a * math.sin(th) + b * math.cos(th)) / k2
                f.write(f"{n} {p} {q} {a!r} {b!r} {ix} {iy} {phi!r} {dth * 2 * math.pi * p!r} {dth * 2 * math.pi * q!r}\n")


if __name__ == "__main__":
    main()
