#!/usr/bin/env python3
"""Generator of csrc/features_generated.cuh: straight-line fp32 code for the point-to-simplex
distances of the Kuhn-split evaluation surface (Algorithm A1 step 4-b-i).

Run `python gen_features.py` in this directory to rewrite features_generated.cuh (the generated file
is committed; the build does not need to run this script).  The script holds no numerics: it only
enumerates the faces of the Kuhn triangulation and prints the closed form below for each of them.

Closed form used (derivation in DESIGN.md, "Point-to-simplex distance"):
a face of the Kuhn mesh is a chain  b = c+S_0, c+S_1, ..., c+S_k  (S_0 < S_1 < ... < S_k axis
subsets).  Its chain edges E_i = (spatial step over the axes T_i = S_i \\ S_{i-1}, dose step dl_i) have
mutually orthogonal spatial parts, so the normal equations (V^T V) w = V^T P of PAPER.md:204 are
"diagonal + rank one" and solve in closed form:
    A_i = sum_{a in T_i} h_a^2          lam_i = -(b . step_i)/A_i     w_i = dl_i / A_i
    N   = d_b + sum dl_i lam_i          G1 = 1 + sum dl_i w_i         r = N / G1
    t_i = lam_i - r w_i                 feasible  <=>  1 >= t_1 >= ... >= t_k >= 0
    dist^2 = C + N r                    C = squared distance from the reference point to the spatial
                                            affine hull of the face (depends on the offset only)
Three routines are emitted:
  * gamma_star_gmax   -- the 75 faces that contain the reference voxel itself (C = 0, N = d0,
                         lam in {0,1}):  gamma_star^2 = d0^2 / max feasible G1, no division per face;
  * gamma_owned_min   -- the 26 faces owned by a grid vertex c (= faces whose lowest vertex is c),
                         any offset, with per-face validity (faces that would leave the grid);
  * gamma_owned_argmin -- gamma_owned_min that also returns the foot point (closest-point output, general geometry);
  * gamma_ring_min    -- the 72 faces of the 2x2x2 block of cells around an interior reference voxel that neither
                         contain the voxel (those are the star) nor lie on the block's boundary (those are at least
                         one voxel spacing away): together with the star, everything closer than min_a h_a.  The
                         offsets are compile-time, so lam_i and C are per-geometry constants (gamma_ring_constants,
                         evaluated once on the host in double precision).
"""
import itertools
import os

AX = (1, 2, 4)  # bit masks of x, y, z


def chains():
    """All chains {} < S_1 < ... < S_k (k = 1..3) of axis subsets: the 26-1 = 25 non-vertex faces."""
    out = []
    subsets = range(1, 8)
    for s1 in subsets:
        out.append((s1,))
        for s2 in subsets:
            if s2 != s1 and (s1 & s2) == s1:
                out.append((s1, s2))
                for s3 in subsets:
                    if s3 != s2 and (s2 & s3) == s2:
                        out.append((s1, s2, s3))
    assert len(out) == 25, len(out)
    return out


def vid(o):
    """index of the neighbour at offset o in {-1,0,1}^3 inside the 27-array (x fastest)."""
    return (o[0] + 1) + 3 * (o[1] + 1) + 9 * (o[2] + 1)


def add(o, mask):
    return tuple(o[a] + (1 if mask & AX[a] else 0) for a in range(3))



def emit_select_helpers(w):
    """gamma_min_if<n> / gamma_max_if<n>: best = min / max(best, x) when a_1 >= b_1 && ... && a_n >= b_n.

    The feasibility test of a face is a chain of ordered comparisons (1 >= t_1 >= ... >= t_k >= 0).  Written as C++
    the compiler turns every comparison into an FSETP plus an FSEL on the candidate; here the comparisons feed one
    predicate (setp.ge.and takes the previous predicate as its third operand) that guards a single FMNMX: k + 2
    instructions per face instead of 2k + 3.  NaN operands fail every comparison (ordered compare), which is how faces
    that would leave the grid are rejected (gamma_owned_min)."""
    w("// best = min(best, x) / max(best, x) when every a_i >= b_i: one predicate through a chain of FSETPs (each takes\n")
    w("// the previous predicate as an input) guarding ONE predicated FMNMX; a NaN operand fails its comparison.\n")
    for op in ("min", "max"):
        for n in range(1, 5):
            args = ", ".join("float a%d, float b%d" % (i, i) for i in range(n))
            w("GAMMA_HD void gamma_%s_if%d(float& best, float x, %s)\n{\n" % (op, n, args))
            w("#if defined(__CUDA_ARCH__)\n")
            lines = ["{", ".reg .pred p;", "setp.ge.f32 p, %2, %3;"]
            for i in range(1, n):
                lines.append("setp.ge.and.f32 p, %%%d, %%%d, p;" % (2 + 2 * i, 3 + 2 * i))
            lines.append("@p %s.f32 %%0, %%0, %%1;" % op)
            lines.append("}")
            body = "\\n\\t".join(lines)
            ins = ", ".join(['"f"(x)'] + ['"f"(a%d), "f"(b%d)' % (i, i) for i in range(n)])
            w('    asm("%s" : "+f"(best) : %s);\n' % (body, ins))
            w("#else\n")
            cond = " && ".join("(a%d >= b%d)" % (i, i) for i in range(n))
            w("    if (%s) best = f%sf(best, x);\n" % (cond, op))
            w("#endif\n}\n")
    w("\n")


def emit_star(w):
    w("// The 75 faces of the Kuhn mesh that contain the reference voxel (its star), generated.\n")
    w("// d[27]: (D_e[v+o] - D_r[v]) / dD for o in {-1,0,1}^3, index (ox+1) + 3(oy+1) + 9(oz+1).\n")
    w("// invA[T]: 1 / sum_{a in T} h_a^2 for the 7 axis subsets T.  Returns the largest feasible\n")
    w("// G1 = 1 + |grad|^2 (>= 1: the vertex itself);  gamma_star = |d0| / sqrt(G1max).\n")
    w("GAMMA_HD float gamma_star_gmax(const float (&d)[27], const float (&invA)[8])\n{\n")
    w("    const float d0 = d[13];\n    float gmax = 1.0f;\n")
    edges = {}      # (vidA, T) -> name
    sums = {}       # tuple of edge names -> name
    lines = []

    def edge(a_off, tmask):
        key = (vid(a_off), tmask)
        if key not in edges:
            nm = "e%d_%d" % key
            b_off = add(a_off, tmask)
            lines.append("    const float dl_%s = d[%d] - d[%d];\n" % (nm, vid(b_off), vid(a_off)))
            lines.append("    const float w_%s = dl_%s * invA[%d];\n" % (nm, nm, tmask))
            lines.append("    const float u_%s = d0 * w_%s;\n" % (nm, nm))
            edges[key] = nm
        return edges[key]

    def gsum(names):
        key = tuple(names)
        if key not in sums:
            nm = "s_" + "_".join(names)
            prev = "1.0f" if len(names) == 1 else gsum(names[:-1])
            lines.append("    const float %s = fmaf(dl_%s, w_%s, %s);\n" % (nm, names[-1], names[-1], prev))
            sums[key] = nm
        return sums[key]

    nfeat = 0
    for o in itertools.product((-1, 0), repeat=3):           # owner (lowest) vertex of the face
        neg = sum(AX[a] for a in range(3) if o[a] == -1)     # subset S with c + S = v
        for ch in chains():
            full = (0,) + ch
            if neg not in full:
                continue
            jstar = full.index(neg)
            k = len(ch)
            names = []
            for i in range(1, k + 1):
                names.append(edge(add(o, full[i - 1]), full[i] ^ full[i - 1]))
            G1 = gsum(names)
            u = ["u_" + n for n in names]
            conds = []                                        # (a, b): a >= b
            # cond_0: G1 >= T_1
            conds.append((u[0], "0.0f") if jstar >= 1 else (G1, "-" + u[0]))
            for i in range(1, k):                             # T_i >= T_{i+1}
                if (i <= jstar) == (i + 1 <= jstar):
                    conds.append((u[i], u[i - 1]))
                else:
                    conds.append((G1, "%s - %s" % (u[i - 1], u[i])))
            conds.append((G1, u[k - 1]) if jstar == k else ("0.0f", u[k - 1]))
            lines.append("    // owner (%d,%d,%d) chain %s, reference voxel is chain vertex %d\n"
                         % (o[0], o[1], o[2], "<".join(str(s) for s in full), jstar))
            lines.append("    gamma_max_if%d(gmax, %s, %s);\n" % (len(conds), G1, ", ".join("%s, %s" % c for c in conds)))
            nfeat += 1
    assert nfeat == 74, nfeat       # + the vertex itself = 75
    for ln in lines:
        w(ln)
    w("    return gmax;\n}\n\n")


def emit_owned(w):
    w("// The 26 faces owned by one grid vertex c at integer offset o from the reference voxel\n")
    w("// (vertex, 7 edges, 12 triangles, 6 tetrahedra whose lowest corner is c), generated.\n")
    w("// d[S]:   (D_e[c+S] - D_r[v]) / dD for the 8 corners S (bit0 = +x, bit1 = +y, bit2 = +z);\n")
    w("// lam[T]: -(p . h_T)/A_T, p = o*h;  q[a] = p_a^2;  X[T] (T = 3,5,6,7): squared distance of p's\n")
    w("//         T-components to the line along h_T.\n")
    w("// A face that would leave the grid (its chain steps along an axis a with c_a + 1 outside) must be rejected by the\n")
    w("// caller's lam: lam[T] = NaN for every T that holds such an axis (owned_face_terms) -- N, r and every t_i of the\n")
    w("// face are then NaN and its first comparison fails.\n")
    w("// Returns min(best2, squared distance to every feasible, valid owned face).\n")
    w("GAMMA_HD float gamma_owned_min(const float (&d)[8], const float (&invA)[8], const float (&lam)[8],\n")
    w("                               const float (&q)[3], const float (&X)[8], float best2)\n{\n")
    w("    best2 = fminf(best2, (q[0] + q[1]) + (q[2] + d[0] * d[0]));   // the vertex c itself\n")
    done_e, done_n, done_g, done_c = set(), set(), set(), set()

    def edge(a, b):
        nm = "%d_%d" % (a, b)
        if nm not in done_e:
            w("    const float dl%s = d[%d] - d[%d];\n" % (nm, b, a))
            w("    const float w%s = dl%s * invA[%d];\n" % (nm, nm, a ^ b))
            done_e.add(nm)
        return nm

    def nsum(full):
        nm = "N" + "_".join(str(s) for s in full)
        if nm not in done_n:
            e = edge(full[-2], full[-1])
            prev = "d[0]" if len(full) == 2 else nsum(full[:-1])
            w("    const float %s = fmaf(dl%s, lam[%d], %s);\n" % (nm, e, full[-1] ^ full[-2], prev))
            done_n.add(nm)
        return nm

    def gsum(full):
        nm = "G" + "_".join(str(s) for s in full)
        if nm not in done_g:
            e = edge(full[-2], full[-1])
            prev = "1.0f" if len(full) == 2 else gsum(full[:-1])
            w("    const float %s = fmaf(dl%s, w%s, %s);\n" % (nm, e, e, prev))
            done_g.add(nm)
        return nm

    def cval(ch):
        full = (0,) + ch
        steps = [full[i] ^ full[i - 1] for i in range(1, len(full))]
        terms = ["X[%d]" % t for t in steps if bin(t).count("1") >= 2]
        terms += ["q[%d]" % a for a in range(3) if not (ch[-1] & AX[a])]
        return " + ".join(terms) if terms else None

    for ch in chains():
        full = (0,) + ch
        k = len(ch)
        names = [edge(full[i - 1], full[i]) for i in range(1, k + 1)]
        N, G = nsum(full), gsum(full)
        tag = "_".join(str(s) for s in ch)
        w("    {   // chain %s\n" % "<".join(str(s) for s in full))
        w("        const float r = GAMMA_FDIV(%s, %s);\n" % (N, G))
        ts = []
        for i in range(k):
            w("        const float t%d = fmaf(-r, w%s, lam[%d]);\n" % (i + 1, names[i], full[i + 1] ^ full[i]))
            ts.append("t%d" % (i + 1))
        conds = [("1.0f", "t1")] + [(ts[i], ts[i + 1]) for i in range(k - 1)] + [(ts[-1], "0.0f")]
        c = cval(ch)
        dist = "fmaf(%s, r, %s)" % (N, c) if c else "%s * r" % N
        w("        gamma_min_if%d(best2, %s, %s);\n" % (len(conds), dist, ", ".join("%s, %s" % x for x in conds)))
        w("    }\n")
    w("    return best2;\n}\n")


def emit_owned_arg(w):
    """gamma_owned_argmin: gamma_owned_min that also reports WHERE the minimum is (general geometry: closest point)."""
    w("\n// gamma_owned_min with the foot point: when a face improves best2, loc[a] (a = 0..2) receives the cell-local\n")
    w("// coordinate of the foot along axis a (0..1 from the owner vertex c) and loc[3] the normalised dose of the surface\n")
    w("// there, (D_e(foot) - D_r[v]) / dD.  Same faces, same arithmetic as gamma_owned_min; run once per voxel, on the\n")
    w("// owner vertex that won the search (closest-point output of the general-geometry path).\n")
    w("GAMMA_HD float gamma_owned_argmin(const float (&d)[8], const float (&invA)[8], const float (&lam)[8],\n")
    w("                                  const float (&q)[3], const float (&X)[8], unsigned usable, float best2,\n")
    w("                                  float (&loc)[4])\n{\n")
    w("    {\n        const float dv = (q[0] + q[1]) + (q[2] + d[0] * d[0]);   // the vertex c itself\n")
    w("        if (dv < best2) { best2 = dv; loc[0] = 0.0f; loc[1] = 0.0f; loc[2] = 0.0f; loc[3] = d[0]; }\n    }\n")
    done_e, done_n, done_g = set(), set(), set()
    for s in range(1, 8):
        w("    const bool ok%d = (usable & %du) == %du;\n" % (s, s, s))

    def edge(a, b):
        nm = "%d_%d" % (a, b)
        if nm not in done_e:
            w("    const float dl%s = d[%d] - d[%d];\n" % (nm, b, a))
            w("    const float w%s = dl%s * invA[%d];\n" % (nm, nm, a ^ b))
            done_e.add(nm)
        return nm

    def nsum(full):
        nm = "N" + "_".join(str(s) for s in full)
        if nm not in done_n:
            e = edge(full[-2], full[-1])
            prev = "d[0]" if len(full) == 2 else nsum(full[:-1])
            w("    const float %s = fmaf(dl%s, lam[%d], %s);\n" % (nm, e, full[-1] ^ full[-2], prev))
            done_n.add(nm)
        return nm

    def gsum(full):
        nm = "G" + "_".join(str(s) for s in full)
        if nm not in done_g:
            e = edge(full[-2], full[-1])
            prev = "1.0f" if len(full) == 2 else gsum(full[:-1])
            w("    const float %s = fmaf(dl%s, w%s, %s);\n" % (nm, e, e, prev))
            done_g.add(nm)
        return nm

    def cval(ch):
        full = (0,) + ch
        steps = [full[i] ^ full[i - 1] for i in range(1, len(full))]
        terms = ["X[%d]" % t for t in steps if bin(t).count("1") >= 2]
        terms += ["q[%d]" % a for a in range(3) if not (ch[-1] & AX[a])]
        return " + ".join(terms) if terms else None

    for ch in chains():
        full = (0,) + ch
        k = len(ch)
        names = [edge(full[i - 1], full[i]) for i in range(1, k + 1)]
        N, G = nsum(full), gsum(full)
        w("    {   // chain %s\n" % "<".join(str(s) for s in full))
        w("        const float r = GAMMA_FDIV(%s, %s);\n" % (N, G))
        ts = []
        for i in range(k):
            w("        const float t%d = fmaf(-r, w%s, lam[%d]);\n" % (i + 1, names[i], full[i + 1] ^ full[i]))
            ts.append("t%d" % (i + 1))
        conds = ["ok%d" % ch[-1], "1.0f >= t1"]
        conds += ["%s >= %s" % (ts[i], ts[i + 1]) for i in range(k - 1)]
        conds.append("%s >= 0.0f" % ts[-1])
        c = cval(ch)
        dist = "fmaf(%s, r, %s)" % (N, c) if c else "%s * r" % N
        w("        const float dist = %s;\n" % dist)
        locs = []
        for a in range(3):
            val = "0.0f"
            for i in range(k):
                if (full[i + 1] ^ full[i]) & AX[a]:
                    val = ts[i]
            locs.append("loc[%d] = %s;" % (a, val))
        dose = "d[0]"
        for i in range(k):
            dose = "fmaf(%s, dl%s, %s)" % (ts[i], names[i], dose)
        w("        if ((%s) && dist < best2) { best2 = dist; %s loc[3] = %s; }\n"
          % (" & ".join("(%s)" % x for x in conds), " ".join(locs), dose))
        w("    }\n")
    w("    return best2;\n}\n")


def ring_faces():
    """(owner o, neg mask, chain) of the 72 ring faces, in emission order."""
    out = []
    for o in itertools.product((-1, 0), repeat=3):
        neg = sum(AX[a] for a in range(3) if o[a] == -1)
        for ch in chains():
            full = (0,) + ch
            if neg in full:
                continue                                     # contains the reference voxel: star
            verts = [add(o, s) for s in full]
            if any(all(v[a] == -1 for v in verts) or all(v[a] == 1 for v in verts) for a in range(3)):
                continue                                     # lies in a boundary plane of the block
            out.append((o, neg, ch))
    assert len(out) == 72, len(out)
    return out


def emit_ring(w):
    faces = ring_faces()
    w("\n// Per-geometry constants of gamma_ring_min: lam[neg][T] = (sum of h_a^2 over a in T with o_a = -1) / A_T for the\n")
    w("// owner o (neg = mask of its -1 coordinates) and axis subset T;  C[f] = squared distance from the reference\n")
    w("// voxel to the spatial affine hull of ring face f.\n")
    w("struct GammaRingP {\n    float lam[8][8];\n    float C[72];\n};\n\n")
    w("// hh[a] = (spacing_a / DTA)^2 in double; every axis must be active.\n")
    w("inline void gamma_ring_constants(const double (&hh)[3], GammaRingP& R)\n{\n")
    w("    double lam[8][8], X[8][8], q[8][3];\n")
    w("    for (int neg = 0; neg < 8; ++neg) {\n")
    w("        for (int a = 0; a < 3; ++a) q[neg][a] = (neg >> a) & 1 ? hh[a] : 0.0;\n")
    w("        for (int T = 0; T < 8; ++T) {\n")
    w("            double A = 0.0, s = 0.0;\n")
    w("            for (int a = 0; a < 3; ++a)\n")
    w("                if ((T >> a) & 1) { A += hh[a]; if ((neg >> a) & 1) s += hh[a]; }\n")
    w("            lam[neg][T] = T ? s / A : 0.0;\n")
    w("            X[neg][T] = T ? s * (A - s) / A : 0.0;\n")
    w("            R.lam[neg][T] = (float)lam[neg][T];\n")
    w("        }\n    }\n")
    for f, (o, neg, ch) in enumerate(faces):
        full = (0,) + ch
        steps = [full[i] ^ full[i - 1] for i in range(1, len(full))]
        terms = ["X[%d][%d]" % (neg, t) for t in steps if bin(t).count("1") >= 2]
        terms += ["q[%d][%d]" % (neg, a) for a in range(3) if not (ch[-1] & AX[a])]
        w("    R.C[%d] = (float)(%s);\n" % (f, " + ".join(terms) if terms else "0.0"))
    w("}\n\n")
    w("// The 72 ring faces (12 edges, 36 triangles, 24 tetrahedra), generated.  d[27] and invA as in gamma_star_gmax.\n")
    w("// Returns min(best2, squared distance to every feasible ring face).\n")
    w("GAMMA_HD float gamma_ring_min(const float (&d)[27], const float (&invA)[8], const GammaRingP& R, float best2)\n{\n")
    done_e, done_n, done_g = set(), set(), set()

    def edge(a_off, tmask):
        nm = "%d_%d" % (vid(a_off), tmask)
        if nm not in done_e:
            w("    const float dl%s = d[%d] - d[%d];\n" % (nm, vid(add(a_off, tmask)), vid(a_off)))
            w("    const float w%s = dl%s * invA[%d];\n" % (nm, nm, tmask))
            done_e.add(nm)
        return nm

    def chain_edges(o, full):
        return [edge(add(o, full[i - 1]), full[i] ^ full[i - 1]) for i in range(1, len(full))]

    def nsum(o, neg, full):
        nm = "N%d_" % vid(o) + "_".join(str(s) for s in full)
        if nm not in done_n:
            e = chain_edges(o, full)[-1]
            prev = "d[%d]" % vid(o) if len(full) == 2 else nsum(o, neg, full[:-1])
            w("    const float %s = fmaf(dl%s, R.lam[%d][%d], %s);\n" % (nm, e, neg, full[-1] ^ full[-2], prev))
            done_n.add(nm)
        return nm

    def gsum(o, full):
        nm = "G%d_" % vid(o) + "_".join(str(s) for s in full)
        if nm not in done_g:
            e = chain_edges(o, full)[-1]
            prev = "1.0f" if len(full) == 2 else gsum(o, full[:-1])
            w("    const float %s = fmaf(dl%s, w%s, %s);\n" % (nm, e, e, prev))
            done_g.add(nm)
        return nm

    for f, (o, neg, ch) in enumerate(faces):
        full = (0,) + ch
        k = len(ch)
        names = chain_edges(o, full)
        N, G = nsum(o, neg, full), gsum(o, full)
        w("    {   // face %d: owner (%d,%d,%d) chain %s\n" % (f, o[0], o[1], o[2], "<".join(str(s) for s in full)))
        w("        const float r = GAMMA_FDIV(%s, %s);\n" % (N, G))
        ts = []
        for i in range(k):
            w("        const float t%d = fmaf(-r, w%s, R.lam[%d][%d]);\n" % (i + 1, names[i], neg, full[i + 1] ^ full[i]))
            ts.append("t%d" % (i + 1))
        conds = [("1.0f", "t1")] + [(ts[i], ts[i + 1]) for i in range(k - 1)] + [(ts[-1], "0.0f")]
        w("        gamma_min_if%d(best2, fmaf(%s, r, R.C[%d]), %s);\n"
          % (len(conds), N, f, ", ".join("%s, %s" % x for x in conds)))
        w("    }\n")
    w("    return best2;\n}\n")


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    path = os.path.join(here, "features_generated.cuh")
    with open(path, "w") as f:
        w = f.write
        w("// GENERATED by gen_features.py -- do not edit by hand.\n")
        w("// Point-to-simplex distances on the Kuhn-split evaluation surface (PAPER.md:187, 204-209),\n")
        w("// closed form for chains of orthogonal steps; see gen_features.py and DESIGN.md.\n")
        w("#pragma once\n#include <math.h>\n")
        w("#if defined(__CUDACC__)\n#define GAMMA_HD __host__ __device__ __forceinline__\n#else\n#define GAMMA_HD inline\n#endif\n")
        w("// N / G with G >= 1: one MUFU.RCP and one FMUL (relative error ~1e-7; __fdividef adds range fix-ups\n")
        w("// that G >= 1 never needs).\n")
        w("#if defined(__CUDA_ARCH__)\n__device__ __forceinline__ float gamma_fdiv(float a, float b)\n{\n"
          "    float r;\n    asm(\"rcp.approx.ftz.f32 %0, %1;\" : \"=f\"(r) : \"f\"(b));\n    return a * r;\n}\n"
          "#define GAMMA_FDIV(a, b) gamma_fdiv((a), (b))\n#else\n#define GAMMA_FDIV(a, b) ((a) / (b))\n#endif\n\n")
        emit_select_helpers(w)
        emit_star(w)
        emit_owned(w)
        emit_owned_arg(w)
        emit_ring(w)
    print("wrote", path)


if __name__ == "__main__":
    main()
