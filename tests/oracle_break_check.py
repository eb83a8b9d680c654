"""Mutation check of the oracle pins (run by hand: `python tests/oracle_break_check.py`, about a minute).

Applies each deliberate break to a scratch copy of oracle/hpmc_oracle.c in place, rebuilds the oracle, runs the pin tests
named beside it and prints which fail; the source is restored afterwards.  Every break must be caught by at least one test
(the results are quoted in the docstrings of tests/test_oracle_moves.py).  Touches only oracle/ and tests/.
"""
import subprocess
import sys
breaks = [
 ("half angle 3d", "        double h = 0.5 * (double)theta;\n        double sh = sin(h);", "        double h = (double)theta;\n        double sh = sin(h);"),
 ("rho=1", "double rho = sqrt(1.0 - z * z);", "double rho = 1.0;"),
 ("left product", "quat_mul(qd, dq, qn);", "quat_mul(dq, qd, qn);"),
 ("2d sin(2h)", "dq[0] = cos(h); dq[1] = 0.0; dq[2] = 0.0; dq[3] = sin(h);", "dq[0] = cos(h); dq[1] = 0.0; dq[2] = 0.0; dq[3] = sin(2 * h);"),
 ("FY i instead of i+1", "(uint64_t)blk[word & 3] * (uint64_t)(i + 1)", "(uint64_t)blk[word & 3] * (uint64_t)(i)"),
 ("shift all from r[0]", "s->w_f[k] * orc_u01(r[k])", "s->w_f[k] * orc_u01(r[0])"),
 ("shift half range", "s->w_f[k] * orc_u01(r[k])", "s->w_f[k] * 0.5f * orc_u01(r[k])"),
]
good = open('oracle/hpmc_oracle.c').read()
ok = True
for name, a, b in breaks:
    assert a in good, name
    open('oracle/hpmc_oracle.c','w').write(good.replace(a, b))
    subprocess.check_call([sys.executable, 'oracle/build.py'], stdout=subprocess.DEVNULL)
    r = subprocess.run([sys.executable, '-m', 'pytest', 'tests/test_oracle_moves.py', '-q', '--no-header', '-p', 'no:cacheprovider'], capture_output=True, text=True)
    failed = [l for l in r.stdout.splitlines() if l.startswith('FAILED')]
    ok = ok and len(failed) > 0
    print(name, '->', len(failed), 'failed:', [f.split('::')[1].split(' ')[0] for f in failed])
open('oracle/hpmc_oracle.c','w').write(good)
subprocess.check_call([sys.executable, 'oracle/build.py'], stdout=subprocess.DEVNULL)
sys.exit(0 if ok else 1)
