"""Writes gint_kstep_dispatch.inc: the inline-PTX bodies of the k-step dispatch of gint_contract_kernel<0>.

One k-step (4 mesh points) of a 32x32 tile issues a DMMA for every fragment pair (i, j) whose rows AND columns hold
an in-sphere point (4-bit masks ra, ca).  C++ `switch` statements over the 225 patterns are lowered by nvcc to
compare trees; PTX `brx.idx` gives ONE indexed jump (SASS BRX) into straight-line code for exactly the pattern.
Operand numbering of the asm statement: %0..%31 accumulators acc[i][j][h] at (4 i + j) 2 + h, %32..%35 a0..a3,
%36..%39 b0..b3, %40 key.

    python gen_kstep_dispatch.py        # rewrites gint_kstep_dispatch.inc next to this file
"""
import os


def mma(i, j):
    c0, c1 = (4 * i + j) * 2, (4 * i + j) * 2 + 1
    return '"mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%%%d,%%%d}, {%%%d}, {%%%d}, {%%%d,%%%d};\\n\\t"' % (
        c0, c1, 32 + i, 36 + j, c0, c1)


def table(name, n, live):
    labels = ", ".join(("%s%d" % (name, k)) if live(k) else (name + "DONE") for k in range(n))
    return ['"%sTBL: .branchtargets %s;\\n\\t"' % (name, labels), '"brx.idx.uni %%40, %sTBL;\\n\\t"' % name]


def rect():
    out = ['"{\\n\\t"'] + table("KR", 256, lambda k: (k & 15) and (k >> 4))
    for key in range(256):
        ra, ca = key & 15, key >> 4
        if not ra or not ca:
            continue
        out.append('"KR%d:\\n\\t"' % key)
        for i in range(4):
            for j in range(4):
                if (ra >> i) & 1 and (ca >> j) & 1:
                    out.append(mma(i, j))
        out.append('"bra.uni KRDONE;\\n\\t"')
    out.append('"KRDONE:\\n\\t}\\n"')
    return out


def diag():
    out = ['"{\\n\\t"'] + table("KD", 16, lambda k: k != 0)
    for ra in range(1, 16):
        out.append('"KD%d:\\n\\t"' % ra)
        for i in range(4):
            for j in range(i, 4):
                if (ra >> i) & 1 and (ra >> j) & 1:
                    out.append(mma(i, j))
        out.append('"bra.uni KDDONE;\\n\\t"')
    out.append('"KDDONE:\\n\\t}\\n"')
    return out


def run_block(name, tblname, key, a_frags, b_frags, pairs, diag):
    """One pattern of a RUN of consecutive k-steps (1 KB apart in the chunks).  The DMMAs of a k-step go row fragment by
    row fragment; as soon as the DMMAs of row fragment i are issued, its A operand register is reloaded for the next
    k-step (rolling reload: no second A set), and the B operands alternate between two register sets (the B fragments
    are read by every row).  A single warp still keeps the FP64 tensor pipe busy by itself, with 24 operand registers
    instead of 32.  Diagonal tiles (B = A) need no second set at all: a_i is dead once row i is done (rows r <= i
    are the only readers of a_i as a B operand).
    Operands: %0..%31 accumulators, %32 / %33 shared-memory byte addresses of the lane's A / B element of the first
    k-step, %34 number of k-steps, %35 pattern."""
    L = name + str(key)
    o = ['"%s:\\n\\t"' % L]

    def ld_a(pred, i, off):
        return '"%sld.shared.f64 a%d, [pa+%d];\\n\\t"' % (pred, i, 256 * i + off)

    def ld_b(pred, prefix, off):
        return ['"%sld.shared.f64 %sb%d, [pb+%d];\\n\\t"' % (pred, prefix, j, 256 * j + off) for j in b_frags]

    def step(bprefix, next_off):
        out = []
        for i in a_frags:
            for (pi, j) in pairs:
                if pi != i:
                    continue
                c0, c1 = (4 * i + j) * 2, (4 * i + j) * 2 + 1
                bop = ("a%d" % j) if diag else ("%sb%d" % (bprefix, j))
                out.append('"mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%%%d,%%%d}, {a%d}, {%s}, {%%%d,%%%d};\\n\\t"' % (c0, c1, i, bop, c0, c1))
            out.append(ld_a("@p ", i, next_off))
        return out

    for i in a_frags:
        o.append(ld_a("", i, 0))
    o += ld_b("", "", 0)
    o.append('"%sL:\\n\\t"' % L)
    o.append('"setp.gt.u32 p, n, 1;\\n\\t"')
    o += ld_b("@p ", "n", 1024)
    o += step("", 1024)
    o.append('"@!p bra.uni %sDONE;\\n\\t"' % name)
    o.append('"setp.gt.u32 p, n, 2;\\n\\t"')
    o += ld_b("@p ", "", 2048)
    o += step("n", 2048)
    o.append('"add.u32 pa, pa, 2048;\\n\\t"')
    if b_frags:
        o.append('"add.u32 pb, pb, 2048;\\n\\t"')
    o.append('"sub.u32 n, n, 2;\\n\\t"')
    o.append('"@p bra.uni %sL;\\n\\t"' % L)
    o.append('"bra.uni %sDONE;\\n\\t"' % name)
    return o


RUN_HEAD = ['"{\\n\\t"', '".reg .f64 a<4>, b<4>, nb<4>;\\n\\t"', '".reg .pred p;\\n\\t"', '".reg .u32 pa, pb, n;\\n\\t"',
            '"mov.u32 pa, %32;\\n\\t"', '"mov.u32 pb, %33;\\n\\t"', '"mov.u32 n, %34;\\n\\t"']


def rect_runs():
    """off-diagonal tile, all four row fragments active (97 % of the off-diagonal DMMAs): pattern = column mask ca"""
    out = list(RUN_HEAD)
    labels = ", ".join("RR%d" % k if k else "RRDONE" for k in range(16))
    out += ['"RRTBL: .branchtargets %s;\\n\\t"' % labels, '"brx.idx.uni %35, RRTBL;\\n\\t"']
    for ca in range(1, 16):
        cols = [j for j in range(4) if (ca >> j) & 1]
        out += run_block("RR", "RRTBL", ca, [0, 1, 2, 3], cols, [(i, j) for i in range(4) for j in cols], False)
    out.append('"RRDONE:\\n\\t}\\n"')
    return out


def diag_runs():
    """diagonal tile (row group == column group, so B = A): pattern = fragment mask ra, pairs i <= j"""
    out = list(RUN_HEAD)
    labels = ", ".join("DR%d" % k if k else "DRDONE" for k in range(16))
    out += ['"DRTBL: .branchtargets %s;\\n\\t"' % labels, '"brx.idx.uni %35, DRTBL;\\n\\t"']
    for ra in range(1, 16):
        fr = [i for i in range(4) if (ra >> i) & 1]
        out += run_block("DR", "DRTBL", ra, fr, [], [(i, j) for i in fr for j in fr if i <= j], True)
    out.append('"DRDONE:\\n\\t}\\n"')
    return out


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "gint_kstep_dispatch.inc"), "w") as f:
        f.write("// GENERATED by gen_kstep_dispatch.py -- do not edit.  Inline-PTX bodies of the k-step dispatch\n")
        f.write("// (brx.idx jump table over the fragment-activity patterns; see gint_kernels.cu).\n")
        f.write("#define GINT_KSTEP_RECT_ASM \\\n    " + " \\\n    ".join(rect()) + "\n\n")
        f.write("#define GINT_KSTEP_DIAG_ASM \\\n    " + " \\\n    ".join(diag()) + "\n\n")
        f.write("#define GINT_RUN_RECT_ASM \\\n    " + " \\\n    ".join(rect_runs()) + "\n\n")
        f.write("#define GINT_RUN_DIAG_ASM \\\n    " + " \\\n    ".join(diag_runs()) + "\n")


if __name__ == "__main__":
    main()
