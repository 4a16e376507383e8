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


def _common_deps():
    return glob.glob(os.path.join(CSRC, '*.cuh')) + glob.glob(os.path.join(CSRC, '*.h')) + \
        glob.glob(os.path.join(HERE, '..', 'include', '*.h')) + [os.path.abspath(__file__)]


def _deps(src):
    """Files whose change must recompile `src`: the hand-written headers, and for a per-process unit the generated
    headers it includes (one level of #include "..." inside csrc/generated/)."""
    out = [src] + _common_deps()
    todo = [src]
    while todo:
        f = todo.pop()
        if os.path.dirname(f) != os.path.join(CSRC, 'generated'):
            continue
        with open(f) as fh:
            for line in fh:
                if line.startswith('#include "') and '/' not in line.split('"')[1]:
                    inc = os.path.join(CSRC, 'generated', line.split('"')[1])
                    if os.path.exists(inc) and inc not in out:
                        out.append(inc)
                        todo.append(inc)
    return out


def _obj(src):
    return os.path.join(OBJDIR, os.path.basename(src)[:-3] + '.o')


def _stale(src):
    obj = _obj(src)
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(f) > t for f in _deps(src))


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return not any(_stale(s) or os.path.getmtime(_obj(s)) > t for s in sources())


def _common_deps():
    return glob.glob(os.path.join(CSRC, '*.cuh')) + glob.glob(os.path.join(CSRC, '*.h')) + \
        glob.glob(os.path.join(HERE, '..', 'include', '*.h')) + [os.path.abspath(__file__)]


def _deps(src):
    """Files whose change must recompile `src`: the hand-written headers, and for a per-process unit the generated
    headers it includes (one level of #include "..." inside csrc/generated/)."""
    out = [src] + _common_deps()
    todo = [src]
    while todo:
        f = todo.pop()
        if os.path.dirname(f) != os.path.join(CSRC, 'generated'):
            continue
        with open(f) as fh:
            for line in fh:
                if line.startswith('#include "') and '/' not in line.split('"')[1]:
                    inc = os.path.join(CSRC, 'generated', line.split('"')[1])
                    if os.path.exists(inc) and inc not in out:
                        out.append(inc)
                        todo.append(inc)
    return out


def _obj(src):
    return os.path.join(OBJDIR, os.path.basename(src)[:-3] + '.o')


def _stale(src):
    obj = _obj(src)
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(f) > t for f in _deps(src))


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return not any(_stale(s) or os.path.getmtime(_obj(s)) > t for s in sources())


def _compile(src):
    obj = _obj(src)
    cmd = ['nvcc'] + NVCC_FLAGS + ['-c', src, '-o', obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log = r.stdout + r.stderr
    with open(obj[:-2] + '.ptxas.log', 'w') as f:
        f.write(' '.join(cmd) + '\n' + log)
    if r.returncode != 0:
        raise RuntimeError('nvcc failed for %s:\n%s' % (src, log))
    return obj, log


def build(force=False, verbose=False):
    """Recompiles the translation units whose sources or headers changed, then links."""
    if not force and up_to_date():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    todo = [s for s in sources() if force or _stale(s)]
    with ThreadPoolExecutor(max_workers=max(1, min(8, os.cpu_count() or 1))) as ex:
        res = list(ex.map(_compile, todo))
    if verbose:
        for _, log in res:
            sys.stdout.write(log)
    cmd = ['nvcc', '-shared', '-o', LIB] + [_obj(s) for s in sources()] + \
        ['-gencode', 'arch=compute_100a,code=sm_100a']
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError('link failed:\n' + r.stdout + r.stderr)
    return LIB


if __name__ == '__main__':
    print(build(force='--force' in sys.argv, verbose='--verbose' in sys.argv))
