#!/usr/bin/env python
"""Mutation sweep over the ORACLE: are its pins tight?  (TEST INFRASTRUCTURE, not collected by pytest.)

    python tests/mutation_sweep.py FIRST_LINE LAST_LINE SEED NMAX [ops]

Draws NMAX single-token mutants of oracle/hydro_oracle.cpp in the given line range -- a numeric literal x 1.5 (an integer
+ 1), a binary + or - flipped; with a fifth argument the other operators instead (* /, < <=, > >=, && ||, == !=) --, builds
each in a scratch copy of oracle/ + tests/ under /tmp and runs the `-m "not gpu"` oracle tests on it.  A mutant that passes
them all is printed as SURVIVED: it is either equivalent (array sizes, overwritten initial values, clamps that never act) or
a hole in the pins (DESIGN.md 4 lists the pins that came out of the sweeps of round 2: lines 80-570, seeds 7, 11 and 21).
Nothing here touches the CUDA path.  ~10 s per mutant on 8 cores.
"""
import os, re, shutil, subprocess, sys, time, random
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = ROOT + '/oracle/hydro_oracle.cpp'
lines = open(SRC).read().split('\n')
LO, HI = int(sys.argv[1]), int(sys.argv[2])
random.seed(int(sys.argv[3]) if len(sys.argv) > 3 else 1)
NMAX = int(sys.argv[4]) if len(sys.argv) > 4 else 150
cands = []
num = re.compile(r'(?<![\w.])(\d+\.\d*(?:[eE][-+]?\d+)?|\d+(?:[eE][-+]?\d+)|\d+)(?![\w.])')
for ln in range(LO - 1, HI):
    code = lines[ln].split('//')[0]
    if not code.strip() or code.strip().startswith(('#', '*', '/*')): continue
    for m in num.finditer(code):
        tok = m.group(1)
        # skip array sizes / template ints that only index
        cands.append((ln, m.start(1), m.end(1), tok, 'num'))
    for m in re.finditer(r' ([-+]) ', code):
        cands.append((ln, m.start(1), m.end(1), m.group(1), 'op'))
    if len(sys.argv) > 5:
        for m in re.finditer(r' (\*|/|<=|>=|<|>|&&|\|\||==|!=) ', code):
            cands.append((ln, m.start(1), m.end(1), m.group(1), 'op2'))
random.shuffle(cands)
if len(sys.argv) > 5: cands = [c for c in cands if c[4] == 'op2']
cands = cands[:NMAX]
W = '/tmp/mutsweep_%d' % os.getpid()
surv = []
t0 = time.time()
for n, (ln, a, b, tok, kind) in enumerate(sorted(cands)):
    if kind == 'num':
        if re.fullmatch(r'\d+', tok): new = str(int(tok) + 1)
        else: new = repr(float(tok) * 1.5 + (0.25 if float(tok) == 0 else 0))
    elif kind == 'op': new = '-' if tok == '+' else '+'
    else: new = {'*': '/', '/': '*', '<=': '<', '>=': '>', '<': '<=', '>': '>=', '&&': '||', '||': '&&', '==': '!=', '!=': '=='}[tok]
    mut = lines[:]
    mut[ln] = mut[ln][:a] + new + mut[ln][b:]
    shutil.rmtree(W, ignore_errors=True); os.makedirs(W)
    for d in ('oracle', 'tests', 'paper_1511_02137_b200', 'include'):
        shutil.copytree(ROOT + '/' + d, W + '/' + d, ignore=shutil.ignore_patterns('*.so', '__pycache__', 'build', 'run_cfg*.npz'))
    shutil.copy(ROOT + '/bench.py', W); shutil.copy(ROOT + '/__graft_entry__.py', W)
    open(W + '/oracle/hydro_oracle.cpp', 'w').write('\n'.join(mut))
    try:
      r = subprocess.run([sys.executable, '-m', 'pytest', 'tests/test_oracle_scalar.py', 'tests/test_oracle_grid.py', 'tests/test_oracle_riemann.py',
                        'tests/test_oracle_weno5.py', 'tests/test_oracle_limiter.py', 'tests/test_oracle_deposit.py', '-x', '-q', '-m', 'not gpu',
                        '-p', 'no:cacheprovider'], cwd=W, capture_output=True, text=True, timeout=300)
    except subprocess.TimeoutExpired:
        print('killed(timeout) L%d %r -> %r' % (ln + 1, tok, new), flush=True); continue
    tail = r.stdout.strip().split('\n')[-1] if r.stdout.strip() else r.stderr[-100:]
    status = 'SURVIVED' if r.returncode == 0 else 'killed'
    first = ''
    mm = re.search(r'FAILED (\S+)', r.stdout)
    if mm: first = mm.group(1).split('::')[-1]
    elif r.returncode != 0: first = 'error/compile'
    print('%s L%d %r -> %r | %s | %s' % (status, ln + 1, tok, new, lines[ln].strip()[:70], first), flush=True)
    if r.returncode == 0: surv.append((ln + 1, tok, new))
print('survivors', len(surv), 'of', len(cands), 'in %.0f s' % (time.time() - t0))
for s in surv: print(s, lines[s[0] - 1].strip()[:100])
