"""Mutation check of the oracle's pins (no GPU).

Each entry below is ONE plausible mistake in oracle/sws_oracle.c (a dropped term, a wrong sign or
index, a transposed operand, a wrong image term), written as an exact text replacement, together with
the pin that must catch it.  The test compiles the mutated copy into a scratch directory (the oracle
loader honours SWS_ORACLE_SRC / SWS_ORACLE_LIBDIR), runs that pin in a subprocess and requires it to
FAIL; a control run with the unmutated source in the same harness must pass every pin named here.
A pattern that no longer occurs exactly once in the source fails the test too, so the list cannot rot.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
SRC = ROOT / "oracle" / "sws_oracle.c"
PINS = "tests/test_oracle_pins.py"
GREEN = "tests/test_oracle_green.py"
JFNK = "tests/test_oracle_jfnk.py"

# (name, old text, new text, pin expected to fail)
MUTANTS = [
    # --- the integral-equation row the residual returns (eq. (12)) ---
    ("E2_row: sign of the K1 sum",
     "weight(p, i, j) * ((f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1",
     "weight(p, i, j) * (-(f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1",
     f"{PINS}::test_P1b_residual_row_is_eq12_with_its_printed_signs"),
    ("E2_row: K1 sum dropped",
     "weight(p, i, j) * ((f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1",
     "weight(p, i, j) * (0 * (f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1",
     f"{GREEN}::test_PG2_residual_row_obeys_greens_identity"),
    ("E2_row: '- x_i + x*' dropped from the K1 density",
     "weight(p, i, j) * ((f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1",
     "weight(p, i, j) * ((f->phi[AT(i, j)] - ps) * K1",
     f"{GREEN}::test_PG2_residual_row_obeys_greens_identity"),
    ("E2_row: sign of the K2 sum",
     "+ f->zeta_x[AT(i, j)] * K2 - zxs * S2);",
     "- f->zeta_x[AT(i, j)] * K2 - zxs * S2);",
     f"{GREEN}::test_PG2_residual_row_obeys_greens_identity"),
    ("E2_row: S2 subtraction not undone by +zeta_x* I",
     "- sum - zxs * I_S2;",
     "- sum + zxs * I_S2;",
     f"{PINS}::test_P7_tilted_plane"),
    ("E2_row: pi instead of 2 pi",
     "return 2 * PI_R * (ps - xs) + (REAL)p->eps",
     "return PI_R * (ps - xs) + (REAL)p->eps",
     f"{GREEN}::test_PG2_residual_row_obeys_greens_identity"),
    ("E2_row: sign of the source term",
     "return 2 * PI_R * (ps - xs) + (REAL)p->eps",
     "return 2 * PI_R * (ps - xs) - (REAL)p->eps",
     f"{PINS}::test_source_term_at_flat_state"),
    ("E2_row: (zeta*+1)^2 -> zeta*^2 + 1 in the source term",
     "- sum - zxs * I_S2;",
     "- sum - zxs * I_S2 + (REAL)p->eps * (1 / sqrt(xs * xs + ys * ys + zs * zs + 1) - 1 / sqrt(xs * xs + ys * ys + (zs + 1) * (zs + 1)));",
     f"{PINS}::test_PH_source_term_is_harmonic_and_centred_at_minus_one"),
    # --- the parallel routine the term-by-term pins look at ---
    ("E2_terms: sign of the K1 sum",
     "s1 += w * (f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1;",
     "s1 -= w * (f->phi[AT(i, j)] - ps - f->x[i] + xs) * K1;",
     f"{GREEN}::test_PG1_double_layer_sum_obeys_greens_identity"),
    ("E2_terms no longer tied to the row",
     "out[2] = s1; out[3] = s2; out[4] = s3;",
     "out[2] = s1; out[3] = s2 * (REAL)1.0000001; out[4] = s3;",
     f"{PINS}::test_e2_terms_tie_to_residual_row"),
    # --- pair kernels (L107, L109, L169-172) ---
    ("K1 image denominator as printed (y - y*)^2, the garbled L107",
     "REAL Rp2 = ddx * ddx + dp * dp + dz * dz;",
     "REAL Rp2 = ddx * ddx + dm * dm + dz * dz;",
     f"{PINS}::test_P1_full_plane_identity"),
    ("K1 image numerator with (y - y*)",
     "+ (dz - ddx * zeta_x - dp * zeta_y) / (Rp2 * Rp);",
     "+ (dz - ddx * zeta_x - dm * zeta_y) / (Rp2 * Rp);",
     f"{PINS}::test_P1_full_plane_identity"),
    ("K1 numerator: zeta_x and zeta_y transposed",
     "*K1 = (dz - ddx * zeta_x - dm * zeta_y) / (Rm2 * Rm)",
     "*K1 = (dz - ddx * zeta_y - dm * zeta_x) / (Rm2 * Rm)",
     f"{PINS}::test_P2_gauss_flux"),
    ("K1 numerator: sign of zeta - zeta*",
     "*K1 = (dz - ddx * zeta_x - dm * zeta_y) / (Rm2 * Rm)",
     "*K1 = (-dz - ddx * zeta_x - dm * zeta_y) / (Rm2 * Rm)",
     f"{PINS}::test_P2_gauss_flux"),
    ("S2 image: sign of B",
     "+ 1 / sqrt(A * ddx * ddx - B * ddx * dp + C * dp * dp);",
     "+ 1 / sqrt(A * ddx * ddx + B * ddx * dp + C * dp * dp);",
     f"{PINS}::test_P1_full_plane_identity"),
    ("S2: A and C swapped",
     "*S2 = 1 / sqrt(A * ddx * ddx + B * ddx * dm + C * dm * dm)",
     "*S2 = 1 / sqrt(C * ddx * ddx + B * ddx * dm + A * dm * dm)",
     f"{PINS}::test_P1_full_plane_identity"),
    ("K2: image term dropped",
     "*K2 = 1 / Rm + 1 / Rp;",
     "*K2 = 1 / Rm;",
     f"{PINS}::test_P1_full_plane_identity"),
    # --- closed-form I (eq. (23), reading Q5) ---
    ("I: sqrt(A) and sqrt(C) swapped in the antiderivative",
     "if (t != 0) g += (t / sqrt(A)) * asinh(",
     "if (t != 0) g += (t / sqrt(C)) * asinh(",
     f"{PINS}::test_P5_box_integral_matches_quadrature"),
    ("I: image box dropped",
     "+ box_integral(A, B, C, xa - xs, xb - xs, -(yb + ys), -(ya + ys));",
     "+ 0 * box_integral(A, B, C, xa - xs, xb - xs, -(yb + ys), -(ya + ys));",
     f"{PINS}::test_P5_S2_integral_is_direct_plus_image"),
    ("A, B, C: B = zeta_x* zeta_y* (factor 2 lost)",
     "*A = 1 + zxs * zxs; *B = 2 * zxs * zys; *C = 1 + zys * zys;",
     "*A = 1 + zxs * zxs; *B = zxs * zys; *C = 1 + zys * zys;",
     # (any A, B, C used in both S2 and I still converges -- only more slowly -- so Green's identity cannot
     # see this one; what sees it is that S2 must cancel the singularity of K2 at the target)
     f"{PINS}::test_PS_S2_is_the_singular_part_of_K2"),
    ("A, B, C: A and C from the wrong slopes",
     "*A = 1 + zxs * zxs; *B = 2 * zxs * zys; *C = 1 + zys * zys;",
     "*A = 1 + zys * zys; *B = 2 * zxs * zys; *C = 1 + zxs * zxs;",
     f"{PINS}::test_PS_S2_is_the_singular_part_of_K2"),
    ("A, B, C: sign of B",
     "*A = 1 + zxs * zxs; *B = 2 * zxs * zys; *C = 1 + zys * zys;",
     "*A = 1 + zxs * zxs; *B = -2 * zxs * zys; *C = 1 + zys * zys;",
     f"{PINS}::test_PS_S2_is_the_singular_part_of_K2"),
    ("A, B, C: the row and the term-by-term routine no longer share them",
     "  star_ABC(f, k, l, &A, &B, &C);\n  REAL sum = 0;",
     "  star_ABC(f, k, l, &A, &B, &C); B = B / 2;\n  REAL sum = 0;",
     f"{PINS}::test_e2_terms_tie_to_residual_row"),
    # --- weights, reconstruction, spline, midpoints ---
    ("trapezoid weight: full weight on the first/last column",
     "REAL ci = (i == 0 || i == p->N - 1) ? (REAL)0.5 : (REAL)1;",
     "REAL ci = (REAL)1;",
     f"{PINS}::test_P4_weights_sum_to_area"),
    ("x-trapezoid: dx instead of dx/2",
     "f->zeta[AT(k + 1, l)] = f->zeta[AT(k, l)] + (dx / 2) *",
     "f->zeta[AT(k + 1, l)] = f->zeta[AT(k, l)] + dx *",
     f"{PINS}::test_x_trapezoid_expanded_form"),
    ("spline: wrong sign in the not-a-knot end row",
     "rhs[M - 1] = 2 * (D_(M - 3) - D_(M - 2));",
     "rhs[M - 1] = 2 * (D_(M - 3) + D_(M - 2));",
     f"{PINS}::test_P3_spline_matches_scipy"),
    ("spline: y_1 = 0 row not clamped",
     "rhs[0] = s->clamped_first ? (REAL)0 : 2 * (D_(0) - D_(1));",
     "rhs[0] = s->clamped_first ? D_(0) : 2 * (D_(0) - D_(1));",
     f"{PINS}::test_P3_spline_matches_scipy"),
    ("FD scheme: one-sided end stencil",
     "m[(size_t)(M - 1) * stride] = (3 * F_(M - 1) - 4 * F_(M - 2) + F_(M - 3)) / (2 * h);",
     "m[(size_t)(M - 1) * stride] = (F_(M - 1) - F_(M - 2)) / h;",
     f"{PINS}::test_fd_scheme_exact_on_quadratics"),
    ("midpoint: node k instead of the two-point average",
     "#define STAR(arr, k, l) (((arr)[AT(k, l)] + (arr)[AT((k) + 1, l)]) / 2)",
     "#define STAR(arr, k, l) ((arr)[AT(k, l)])",
     f"{PINS}::test_PJ1_exact_jacobian_reproduces_appendix_B"),
    # --- Bernoulli and radiation rows, ordering ---
    ("E1: zeta*/F instead of zeta*/F^2",
     "REAL F2 = (REAL)p->froude * (REAL)p->froude;",
     "REAL F2 = (REAL)p->froude;",
     f"{PINS}::test_E1_bernoulli_formula"),
    ("E1: sign of the cross term",
     "- 2 * zx * zy * px * py)",
     "+ 2 * zx * zy * px * py)",
     f"{PINS}::test_PB_bernoulli_row_on_exact_tilted_plane_flow"),
    ("E1: phi_x and phi_y transposed",
     "((1 + zx * zx) * py * py + (1 + zy * zy) * px * px",
     "((1 + zx * zx) * px * px + (1 + zy * zy) * py * py",
     f"{PINS}::test_PB_bernoulli_row_on_exact_tilted_plane_flow"),
    ("E1: factor 2 of the cross term lost",
     "- 2 * zx * zy * px * py)",
     "- zx * zy * px * py)",
     f"{PINS}::test_PB_bernoulli_row_on_exact_tilted_plane_flow"),
    ("E1: denominator without zeta_y^2",
     "/ (1 + zx * zx + zy * zy) / 2",
     "/ (1 + zx * zx) / 2",
     f"{PINS}::test_PB_bernoulli_row_on_exact_tilted_plane_flow"),
    ("E4: second derivative taken at the wrong nodes",
     "e[1] = x1 * ((f.phi_x[AT(1, l)] - f.phi_x[AT(0, l)]) / dx)",
     "e[1] = x1 * ((f.phi_x[AT(2, l)] - f.phi_x[AT(1, l)]) / dx)",
     f"{PINS}::test_radiation_rows_and_positions"),
    ("E5: n zeta_1 dropped",
     "e2[0] = x1 * f.zeta_x[AT(0, l)] + n * f.zeta[AT(0, l)];",
     "e2[0] = x1 * f.zeta_x[AT(0, l)];",
     f"{PINS}::test_radiation_rows_and_positions"),
    ("ordering: E2 rows written one slot early (App. A L421)",
     "E[half + (size_t)l * (N + 1) + 2 + k] = E2_row(p, &f, k, l);",
     "E[half + (size_t)l * (N + 1) + 1 + k] = E2_row(p, &f, k, l);",
     f"{PINS}::test_P7_tilted_plane"),
    ("unknown ordering: zeta block read at the phi offset (eq. (18) L149)",
     "const size_t off_zeta = (size_t)(N + 1) * M;",
     "const size_t off_zeta = 0;",
     f"{PINS}::test_x_trapezoid_expanded_form"),
]


def _run(src: Path, libdir: Path, nodes):
    env = dict(os.environ, SWS_ORACLE_SRC=str(src), SWS_ORACLE_LIBDIR=str(libdir), OMP_NUM_THREADS="1")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", *nodes],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    return r.returncode, r.stdout[-1500:] + r.stderr[-500:]


def _mutant(args):
    i, (name, old, new, pin), tmp = args
    text = SRC.read_text()
    if text.count(old) != 1:
        return name, None, f"pattern occurs {text.count(old)} times in sws_oracle.c (want exactly 1)"
    d = tmp / f"m{i:02d}"
    d.mkdir()
    (d / "sws_oracle.c").write_text(text.replace(old, new))
    rc, out = _run(d / "sws_oracle.c", d, [pin])
    return name, rc, out


def test_control_unmutated_source_passes_every_pin_named_here(tmp_path):
    d = tmp_path / "control"
    d.mkdir()
    (d / "sws_oracle.c").write_text(SRC.read_text())
    rc, out = _run(d / "sws_oracle.c", d, sorted({m[3] for m in MUTANTS}))
    assert rc == 0, out


def test_every_mutant_fails_its_pin(tmp_path):
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        results = list(ex.map(_mutant, [(i, m, tmp_path) for i, m in enumerate(MUTANTS)]))
    survivors = []
    for name, rc, out in results:
        if rc is None:
            survivors.append(f"{name}: {out}")
        elif rc == 0:
            survivors.append(f"{name}: the pin PASSED on the mutant")
        elif rc != 1:                     # 1 = tests failed; anything else = harness / compile error
            survivors.append(f"{name}: pytest exit code {rc}\n{out}")
    assert not survivors, "\n".join(survivors)
    assert len(results) >= 30
