"""Mutation check of the oracle pins (run by hand: `python tests/oracle_break_check.py`, about a minute).

Applies each deliberate break to a scratch copy of oracle/hpmc_oracle.c in place, rebuilds the oracle, runs the pin tests
named beside it and prints which fail; the source is restored afterwards.  Every break must be caught by at least one test
(the results are quoted in the docstrings of tests/test_oracle_moves.py; the rounded-shape breaks run tests/test_oracle_rounded.py).  Touches only oracle/ and tests/.
"""
import subprocess
import sys
# (name, text in hpmc_oracle.c, its replacement[, test file]) -- test file defaults to tests/test_oracle_moves.py
breaks = [
 ("half angle 3d", "        double h = 0.5 * (double)theta;\n        double sh = sin(h);", "        double h = (double)theta;\n        double sh = sin(h);"),
 ("rho=1", "double rho = sqrt(1.0 - z * z);", "double rho = 1.0;"),
 ("left product", "quat_mul(qd, dq, qn);", "quat_mul(dq, qd, qn);"),
 ("2d sin(2h)", "dq[0] = cos(h); dq[1] = 0.0; dq[2] = 0.0; dq[3] = sin(h);", "dq[0] = cos(h); dq[1] = 0.0; dq[2] = 0.0; dq[3] = sin(2 * h);"),
 ("FY i instead of i+1", "(uint64_t)blk[word & 3] * (uint64_t)(i + 1)", "(uint64_t)blk[word & 3] * (uint64_t)(i)"),
 ("shift all from r[0]", "s->w_f[k] * orc_u01(r[k])", "s->w_f[k] * orc_u01(r[0])"),
 ("shift half range", "s->w_f[k] * orc_u01(r[k])", "s->w_f[k] * 0.5f * orc_u01(r[k])"),
 # rounded shapes, caught by tests/test_oracle_rounded.py
 ("rounded: one radius", "return m - 2.0 * s->sweep_r;", "return m - s->sweep_r;", "tests/test_oracle_rounded.py"),
 ("rounded: separating-axis margin instead of the distance", "        m = core_distance(s, r_ab, qa, qb, wa, wb);", "        ;", "tests/test_oracle_rounded.py"),
 ("rounded: no vertex-face pairs", "                if (inside && h < best) best = h;", "                (void)inside;", "tests/test_oracle_rounded.py"),
 ("rounded: no interior edge-edge point", "if (sc > 0.0 && sc < 1.0 && tc > 0.0 && tc < 1.0) {", "if (0) {", "tests/test_oracle_rounded.py"),
 ("rounded: segment clamp dropped", "    if (t > 1.0) t = 1.0;", "", "tests/test_oracle_rounded.py"),
 ("rounded: d_max without the radius", "s->dmax = 2.0 * (rmax + sweep_r);", "s->dmax = 2.0 * rmax;", "tests/test_oracle_rounded.py"),
]
good = open('oracle/hpmc_oracle.c').read()
ok = True
for name, a, b, *rest in breaks:
    test_file = rest[0] if rest else 'tests/test_oracle_moves.py'
    assert a in good, name
    open('oracle/hpmc_oracle.c','w').write(good.replace(a, b))
    subprocess.check_call([sys.executable, 'oracle/build.py'], stdout=subprocess.DEVNULL)
    r = subprocess.run([sys.executable, '-m', 'pytest', test_file, '-q', '--no-header', '-p', 'no:cacheprovider'], capture_output=True, text=True)
    failed = [l for l in r.stdout.splitlines() if l.startswith('FAILED')]
    ok = ok and len(failed) > 0
    print(name, '->', len(failed), 'failed:', [f.split('::')[1].split(' ')[0] for f in failed])
open('oracle/hpmc_oracle.c','w').write(good)
subprocess.check_call([sys.executable, 'oracle/build.py'], stdout=subprocess.DEVNULL)
sys.exit(0 if ok else 1)
