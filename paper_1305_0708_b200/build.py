"""Builds paper_1305_0708_b200/libhg.so (the C-ABI library of include/hg.h) for sm_100a with nvcc.

One translation unit per process (csrc/generated/hg_proc_<pid>.cu) plus csrc/hg_api.cu, compiled in parallel and
linked in-tree.  `python -m paper_1305_0708_b200.build [--force] [--verbose]`.
"""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, 'csrc')
LIB = os.path.join(HERE, 'libhg.so')
OBJDIR = os.path.join(HERE, 'build')

NVCC_FLAGS = ['-gencode', 'arch=compute_100a,code=sm_100a', '-lineinfo', '-O3', '-std=c++17',
              '--expt-relaxed-constexpr', '-Xcompiler', '-fPIC', '-Xptxas', '-v']


def sources():
    return [os.path.join(CSRC, 'hg_api.cu')] + sorted(glob.glob(os.path.join(CSRC, 'generated', 'hg_proc_*.cu')))


def _deps():
    out = sources() + glob.glob(os.path.join(CSRC, '*.cuh')) + glob.glob(os.path.join(CSRC, '*.h')) + \
        glob.glob(os.path.join(CSRC, 'generated', '*.cuh')) + [os.path.join(HERE, '..', 'include', 'hg.h'),
                                                                os.path.abspath(__file__)]
    return out


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(f) <= t for f in _deps())


def _compile(src):
    obj = os.path.join(OBJDIR, os.path.basename(src)[:-3] + '.o')
    cmd = ['nvcc'] + NVCC_FLAGS + ['-c', src, '-o', obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log = r.stdout + r.stderr
    with open(obj[:-2] + '.ptxas.log', 'w') as f:
        f.write(' '.join(cmd) + '\n' + log)
    if r.returncode != 0:
        raise RuntimeError('nvcc failed for %s:\n%s' % (src, log))
    return obj, log


def build(force=False, verbose=False):
    if not force and up_to_date():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    with ThreadPoolExecutor(max_workers=max(1, min(8, os.cpu_count() or 1))) as ex:
        res = list(ex.map(_compile, sources()))
    if verbose:
        for _, log in res:
            sys.stdout.write(log)
    cmd = ['nvcc', '-shared', '-o', LIB] + [o for o, _ in res] + ['-gencode', 'arch=compute_100a,code=sm_100a']
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError('link failed:\n' + r.stdout + r.stderr)
    return LIB


if __name__ == '__main__':
    print(build(force='--force' in sys.argv, verbose='--verbose' in sys.argv))
