"""python -m paper_1309_1720_b200.sass_count  (after a build; needs cuobjdump)

FP64 instructions per cell-step from the SASS of ring_stage_kernel<model, stencil, kind> (whole function =
one pair per thread and tile iteration; no FP64 outside the per-pair body): (DFMA, DMUL, DADD) / 2 per kind.
The table FP64_PER_CELL_STEP of bench.py is this output."""
import collections
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
out = subprocess.run(["cuobjdump", "-sass", os.path.join(HERE, "build", "stream_kernels.o")], capture_output=True, text=True).stdout
fn = None; cnt = collections.defaultdict(collections.Counter)
for line in out.splitlines():
    m = re.search(r"Function : (\S+)", line)
    if m: fn = m.group(1); continue
    m = re.search(r"/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", line)
    if m and fn and "ring_stage_kernel" in fn:
        op = m.group(1).split(".")[0]
        if op in ("DFMA", "DMUL", "DADD", "DSETP"): cnt[fn][op] += 1
def key(fn):
    m = re.search(r"ModelILi(\d)ELi(\d)EEELi(\d)ELi(\d)E", fn)
    return tuple(int(x) for x in m.groups())   # model, variant, stencil, kind
tab = {key(f): c for f, c in cnt.items()}
for (model, var, st, integ, name) in [(0, 0, 0, 'euler', 'cfg1'), (0, 0, 1, 'rk4', 'cfg2/5'), (1, 0, 0, 'rk4', 'cfg3'), (2, 0, 1, 'rk4', 'cfg4')]:
    kinds = [0] if integ == 'euler' else [0, 1, 1, 2]
    ins = sum(sum(tab[(model, var, st, k)].values()) for k in kinds) / 2
    fl = sum(2 * tab[(model, var, st, k)]['DFMA'] + tab[(model, var, st, k)]['DMUL'] + tab[(model, var, st, k)]['DADD'] for k in kinds) / 2
    print(name, (model, st, integ), 'instr', ins, 'flops', fl, {k: dict(tab[(model, var, st, k)]) for k in set(kinds)})
