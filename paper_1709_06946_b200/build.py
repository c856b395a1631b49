"""Build libpse.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, 'csrc')
LIB = os.path.join(HERE, 'libpse.so')
SOURCES = ['tables.cu', 'neighbors.cu', 'realspace.cu', 'wavespace.cu', 'krylov.cu', 'api.cu', 'couplet.cu', 'noalloc.cu']
CUDA_HOME = os.environ.get('CUDA_HOME', '/usr/local/cuda')


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, 'include', 'pse.h')]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile every CUDA source into paper_1709_06946_b200/libpse.so; returns its path."""
    if not force and not _stale():
        return LIB
    nvcc = os.path.join(CUDA_HOME, 'bin', 'nvcc')
    objdir = os.path.join(HERE, 'build')
    os.makedirs(objdir, exist_ok=True)
    flags = ['-O3', '-std=c++17', '-gencode', 'arch=compute_100a,code=sm_100a', '-lineinfo',
             '-Xcompiler', '-fPIC', '-I', os.path.join(ROOT, 'include'), '-I', CSRC]
    if verbose:
        flags += ['-Xptxas', '-v']
    procs = []
    objs = []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace('.cu', '.o'))
        objs.append(obj)
        procs.append((src, subprocess.Popen([nvcc, *flags, '-c', os.path.join(CSRC, src), '-o', obj],
                                            stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for src, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out)
        if p.returncode:
            raise RuntimeError(f'nvcc failed on {src}')
    libdir = os.path.join(CUDA_HOME, 'lib64')
    cmd = [nvcc, '-shared', '-o', LIB, *objs, '-L', libdir, '-lcufft', '-Xlinker', f'-rpath={libdir}']
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode:
        sys.stderr.write(r.stdout)
        raise RuntimeError('link failed')
    return LIB


if __name__ == '__main__':
    print(build(force='--force' in sys.argv, verbose='-v' in sys.argv))
