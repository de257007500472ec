"""Mutation run of the oracle pins (CPU only): every plausible single-line mistake in oracle/gf_oracle.c must
fail at least one test of tests/test_oracle_pins.py.

For each mutant a private copy of oracle/, gf_inputs.py, the pins and tests/golden/ is made in a temporary
directory, ONE line of the C source is replaced, the library is rebuilt there and the pins are run with
``pytest -x``; the run must fail.  The unmutated copy must pass (control).  Nothing of the CUDA path is involved.
The mutants are the mistakes SURVEY.md 8(c) and the round-1 review name: signs of v, missing daggers, wrong
neighbour, dropped trace, omega / subgroup / draw mix-ups, left instead of right multiplication, normalisations,
Philox constants and counter layout, the 24-bit fraction, the unitarity checker's two outputs; a second batch: the
periodic wrap, the site index, the SU(2) embedding, normalisations of a, Coulomb sums, the Philox site key, the plaquette.
"""
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "gf_oracle.c")

# (name, exact source fragment, replacement); every fragment must occur exactly once in gf_oracle.c
MUTANTS = [
    ("v1 sign", "v[1] = -cimag(Kij + Kji);", "v[1] = cimag(Kij + Kji);"),
    ("v2 sign", "v[2] = creal(Kji - Kij);", "v[2] = creal(Kij - Kji);"),
    ("v3 sign", "v[3] = cimag(Kjj - Kii);", "v[3] = cimag(Kii - Kjj);"),
    ("v0 difference instead of sum", "v[0] = creal(Kii + Kjj);", "v[0] = creal(Kii - Kjj);"),
    ("K without the dagger on the backward link", "K[k] += fwd[mu][k] + bd[k];", "K[k] += fwd[mu][k] + bwd[mu][k];"),
    ("K from the forward neighbour", "bwd[mu] = (cd *)link_cptr(U, neighbour(dims, c, mu, -1), mu);\n    }\n    build_K",
     "bwd[mu] = (cd *)link_cptr(U, neighbour(dims, c, mu, +1), mu);\n    }\n    build_K"),
    ("sweep touches the forward neighbour", "bwd[mu] = link_ptr(U, neighbour(dims, c, mu, -1), mu);",
     "bwd[mu] = link_ptr(U, neighbour(dims, c, mu, +1), mu);"),
    ("trace kept in A", "A[0] -= tr; A[4] -= tr; A[8] -= tr;", ""),
    ("factor 2 in A", "A[k] = (u[k] - ud[k]) / (2.0 * I);", "A[k] = (u[k] - ud[k]) / (1.0 * I);"),
    ("forward difference in Delta", "gauge_field_A(link_cptr(U, neighbour(dims, c, mu, -1), mu), Ab);",
     "gauge_field_A(link_cptr(U, neighbour(dims, c, mu, +1), mu), Ab);"),
    ("overrelaxation omega sign", "omega * v[0] + (1.0 - omega) * n,", "omega * v[0] - (1.0 - omega) * n,"),
    ("overrelaxation without the norm", "omega * v[0] + (1.0 - omega) * n,", "omega * v[0] + (1.0 - omega),"),
    ("stochastic: u <= p", "algo == ORACLE_STOCHASTIC && u < p", "algo == ORACLE_STOCHASTIC && u <= p"),
    ("stochastic: a^2 with the wrong a0", "a[0] = 2.0 * a0 * a0 - 1.0;", "a[0] = 2.0 * a0 * a0;"),
    ("subgroup order", "{ { 0, 1 }, { 0, 2 }, { 1, 2 } }", "{ { 0, 1 }, { 1, 2 }, { 0, 2 } }"),
    ("third subgroup not overrelaxed", "oracle_su2_update(v, algo, omega, p, u[k], a);",
     "oracle_su2_update(v, algo, k == 2 ? 1.0 : omega, p, u[k], a);"),
    ("one draw for all three subgroups", "oracle_su2_update(v, algo, omega, p, u[k], a);",
     "oracle_su2_update(v, algo, omega, p, u[0], a);"),
    ("draws assigned in reverse", "oracle_su2_update(v, algo, omega, p, u[k], a);",
     "oracle_su2_update(v, algo, omega, p, u[2 - k], a);"),
    ("K not refreshed between subgroups", "embed_left_multiply(K, sub[k][0], sub[k][1], a);", ""),
    ("E_ij and E_ji exchanged", "const cd Eii = a[0] + I * a[3], Eij = a[2] + I * a[1];",
     "const cd Eii = a[0] + I * a[3], Eij = -a[2] + I * a[1];"),
    ("links multiplied from the wrong side", "mat_mul(g, fwd[mu], tmp);", "mat_mul(fwd[mu], g, tmp);"),
    ("backward link without g dagger", "mat_mul(bwd[mu], gd, tmp);", "mat_mul(bwd[mu], g, tmp);"),
    ("Coulomb leaves the temporal links alone", "for (int mu = 0; mu < 4; ++mu) {\n        mat_mul(g, fwd[mu], tmp);",
     "for (int mu = first_dir(gauge); mu < 4; ++mu) {\n        mat_mul(g, fwd[mu], tmp);"),
    ("Coulomb K over all four directions", "static int first_dir(int gauge) { return gauge == ORACLE_COULOMB ? 1 : 0; }",
     "static int first_dir(int gauge) { (void)gauge; return 0; }"),
    ("F normalisation", "out[t] = sum / ((double)NC * (4 - mu0) * (double)per);", "out[t] = sum / ((double)NC * 4 * (double)per);"),
    ("theta normalisation", "out[t] = sum / ((double)NC * (double)per);\n    }\n}\n\n/* ---",
     "out[t] = sum / ((double)per);\n    }\n}\n\n/* ---"),
    ("parity definition", "return (c[0] + c[1] + c[2] + c[3]) & 1;", "return (c[1] + c[2] + c[3]) & 1;"),
    ("parity order in the fix loop", "oracle_sweep(U, dims, gauge, 0, algo, omega, p, seed, first_counter + 2u * (uint32_t)it);",
     "oracle_sweep(U, dims, gauge, 1, algo, omega, p, seed, first_counter + 2u * (uint32_t)it);"),
    ("theta tested one iteration late", "if (it % check_every == 0 || it == max_iter) {\n            oracle_theta(U, dims, gauge, th);",
     "if (it % check_every == 1 % check_every || it == max_iter) {\n            oracle_theta(U, dims, gauge, th);"),
    ("Philox multiplier", "(uint64_t)0xD2511F53u * c0;", "(uint64_t)0xD2511F55u * c0;"),
    ("Philox key schedule", "k1 += 0xBB67AE85u;", "k1 += 0x9E3779B9u;"),
    ("Philox counter layout", "{ (uint32_t)s, (uint32_t)(s >> 32), half_sweep_counter, 0u };",
     "{ (uint32_t)s, half_sweep_counter, (uint32_t)(s >> 32), 0u };"),
    ("23-bit uniforms", "u[k] = (double)(w[k] >> 8) * (1.0 / 16777216.0);", "u[k] = (double)(w[k] >> 9) * (1.0 / 8388608.0);"),
    ("uniforms from words 1..3", "u[k] = (double)(w[k] >> 8)", "u[k] = (double)(w[k + 1] >> 8)"),
    ("plaquette neighbour", "mat_dagger(link_cptr(U, neighbour(dims, c, nu, +1), mu), d1);",
     "mat_dagger(link_cptr(U, neighbour(dims, c, mu, +1), mu), d1);"),
    ("unitarity: determinant branch dropped", "if (cabs(det - 1) > detmax) detmax = cabs(det - 1);", ""),
    ("unitarity: U U^dagger branch dropped", "if (cabs(P[k]) > dmax) dmax = cabs(P[k]);", "if (cabs(P[k]) > dmax) dmax = 0.0;"),
    ("unitarity: U U instead of U U^dagger", "mat_mul(u, ud, P);\n        P[0] -= 1;", "mat_mul(u, u, P);\n        P[0] -= 1;"),
    ("unitarity: only the first link of a site", "const size_t nlinks = volume(dims) * 4;", "const size_t nlinks = volume(dims);"),
    ("accumulated transformation on the wrong side", "mat_mul(g, Gtot + s * 9, tmp);", "mat_mul(Gtot + s * 9, g, tmp);"),
    ("eq. 3 without the dagger on G(x+mu)", "mat_dagger(G + neighbour(dims, c, mu, +1) * 9, gd);",
     "for (int k = 0; k < 9; ++k) gd[k] = (G + neighbour(dims, c, mu, +1) * 9)[k];"),
    ("eq. 3 with the backward neighbour", "mat_dagger(G + neighbour(dims, c, mu, +1) * 9, gd);",
     "mat_dagger(G + neighbour(dims, c, mu, -1) * 9, gd);"),
    ("slice mask on the wrong axis", "if (slice_active && !slice_active[c[0]]) return;", "if (slice_active && !slice_active[c[3]]) return;"),
    ("periodic wrap: x - mu of the first site lands on itself", "n[mu] = (c[mu] + dir + dims[mu]) % dims[mu];",
     "n[mu] = c[mu] + dir < 0 ? 0 : (c[mu] + dir) % dims[mu];"),
    ("site index with y and z exchanged",
     "return (size_t)c[1] + (size_t)dims[1] * (c[2] + (size_t)dims[2] * (c[3] + (size_t)dims[3] * c[0]));",
     "return (size_t)c[1] + (size_t)dims[1] * (c[3] + (size_t)dims[3] * (c[2] + (size_t)dims[2] * c[0]));"),
    ("E_jj without the conjugation", "Ejj = a[0] - I * a[3];", "Ejj = a[0] + I * a[3];"),
    ("E_ji sign", "const cd Eji = -a[2] + I * a[1]", "const cd Eji = a[2] + I * a[1]"),
    ("g misses the first subgroup", "embed_left_multiply(g, sub[k][0], sub[k][1], a);",
     "if (k > 0) embed_left_multiply(g, sub[k][0], sub[k][1], a);"),
    ("relaxation without the normalisation", "for (int k = 0; k < 4; ++k) a[k] = v[k] / n;", "for (int k = 0; k < 4; ++k) a[k] = v[k];"),
    ("overrelaxation normalised with |v|", "a[k] = w[k] / nw;", "a[k] = w[k] / n;"),
    ("stochastic: one vector component of a^2 not doubled", "a[1] = 2.0 * a0 * a[1];", "a[1] = a0 * a[1];"),
    ("Coulomb Delta over all four directions", "for (int mu = first_dir(gauge); mu < 4; ++mu) {\n        cd Af[9], Ab[9];",
     "for (int mu = 0; mu < 4; ++mu) {\n        cd Af[9], Ab[9];"),
    ("Coulomb F sums the temporal links too", "for (int mu = mu0; mu < 4; ++mu) {\n                const cd *u = link_cptr(U, s, mu);",
     "for (int mu = 0; mu < 4; ++mu) {\n                const cd *u = link_cptr(U, s, mu);"),
    ("Coulomb loop stops on the best slice", "if (th[t] > theta) theta = th[t];", "if (th[t] < theta) theta = th[t];"),
    ("Philox: nine rounds", "for (int round = 0; round < 10; ++round) {", "for (int round = 0; round < 9; ++round) {"),
    ("Philox: second multiplier on c1", "(uint64_t)0xCD9E8D57u * c2;", "(uint64_t)0xCD9E8D57u * c1;"),
    ("Philox: key halves exchanged", "{ (uint32_t)seed, (uint32_t)(seed >> 32) };", "{ (uint32_t)(seed >> 32), (uint32_t)seed };"),
    ("Philox: draws keyed by the per-parity index", "oracle_site_uniforms(seed, half_sweep_counter, (uint64_t)s, u);",
     "oracle_site_uniforms(seed, half_sweep_counter, (uint64_t)(s / 2), u);"),
    ("fix loop: both parities draw with the same counter",
     "oracle_sweep(U, dims, gauge, 1, algo, omega, p, seed, first_counter + 2u * (uint32_t)it + 1u);",
     "oracle_sweep(U, dims, gauge, 1, algo, omega, p, seed, first_counter + 2u * (uint32_t)it);"),
    ("plaquette: last dagger dropped", "mat_dagger(link_cptr(U, s, nu), d2);",
     "for (int k = 0; k < 9; ++k) d2[k] = link_cptr(U, s, nu)[k];"),
    ("plaquette normalisation", "return sum / (6.0 * NC * (double)V);", "return sum / (4.0 * NC * (double)V);"),
    ("update applied in three directions only", "for (int mu = 0; mu < 4; ++mu) {\n        mat_mul(g, fwd[mu], tmp);",
     "for (int mu = 0; mu < 3; ++mu) {\n        mat_mul(g, fwd[mu], tmp);"),
    ("|v| = 0 gives a = 0", "a[0] = 1.0; a[1] = a[2] = a[3] = 0.0;\n        return;", "a[0] = 0.0; a[1] = a[2] = a[3] = 0.0;\n        return;"),
    ("frozen slices never frozen", "if (active[t] && theta_slices[t] < theta_target) { active[t] = 0; frozen_at[t] = it; }",
     "if (active[t] && theta_slices[t] < 0.0) { active[t] = 0; frozen_at[t] = it; }"),
]


def _run_copy(name, old, new):
    tmp = tempfile.mkdtemp(prefix="gf_mutant_")
    try:
        shutil.copytree(os.path.join(ROOT, "oracle"), os.path.join(tmp, "oracle"),
                        ignore=shutil.ignore_patterns("*.so", "__pycache__"))
        shutil.copy(os.path.join(ROOT, "gf_inputs.py"), tmp)
        shutil.copy(os.path.join(ROOT, "tests", "test_oracle_pins.py"), tmp)
        shutil.copytree(os.path.join(ROOT, "tests", "golden"), os.path.join(tmp, "golden"))
        c_file = os.path.join(tmp, "oracle", "gf_oracle.c")
        text = open(c_file).read()
        if old is not None:
            if text.count(old) != 1:
                return name, "fragment occurs %d times in gf_oracle.c (the mutant list is stale)" % text.count(old)
            open(c_file, "w").write(text.replace(old, new))
        env = dict(os.environ, PYTHONPATH=tmp, OMP_NUM_THREADS="1")
        r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "test_oracle_pins.py"],
                           cwd=tmp, env=env, capture_output=True, text=True, timeout=600)
        failed = [l for l in r.stdout.splitlines() if l.startswith("FAILED") or l.startswith("ERROR")]
        if any("CalledProcessError" in l for l in failed):
            return name, "the mutated source does not compile: %s" % failed[0]
        return name, (r.returncode, failed[0] if failed else r.stdout[-300:])
    finally:
        shutil.rmtree(tmp, ignore_errors=True)


def test_every_mutant_of_the_oracle_fails_a_pin():
    jobs = [("control (unmutated)", None, None)] + MUTANTS
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        results = list(ex.map(lambda j: _run_copy(*j), jobs))
    name, res = results[0]
    assert isinstance(res, tuple) and res[0] == 0, "the unmutated copy must pass: %r" % (res,)
    survivors, report = [], []
    for name, res in results[1:]:
        assert isinstance(res, tuple), "%s: %s" % (name, res)
        rc, first = res
        report.append("%-48s -> %s" % (name, first))
        if rc == 0:
            survivors.append(name)
    print("\n".join(report))
    assert not survivors, "mutants that pass every pin: %s" % survivors
