// stl_io.cu -- SURVEY.md 8(f) NEXT-4, the paper's outer I/O shell (host code only): "The code takes
// as input a stereolithography (STL) file and outputs a file that lists the SDF values in a 3D
// grid"; the ASCII facet layout is PAPER.md:278-288.  Vertices are listed
// counter-clockwise seen from outside; the facet normals of the file are ignored,
// sdf_create recomputes them from the vertex order.
#include "common.cuh"
#include <ctype.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

static int read_all(const char *path, unsigned char **buf, size_t *len) {
    FILE *f = fopen(path, "rb");
    if (!f) return SDF_EIO;
    if (fseek(f, 0, SEEK_END) != 0) { fclose(f); return SDF_EIO; }
    long n = ftell(f);
    if (n < 0 || fseek(f, 0, SEEK_SET) != 0) { fclose(f); return SDF_EIO; }
    unsigned char *b = (unsigned char *)malloc((size_t)n + 1);
    if (!b) { fclose(f); return SDF_ENOMEM; }
    if (n > 0 && fread(b, 1, (size_t)n, f) != (size_t)n) { free(b); fclose(f); return SDF_EIO; }
    fclose(f);
    b[n] = 0;
    *buf = b; *len = (size_t)n;
    return SDF_OK;
}

// binary: 80-byte header, uint32 count, then per facet 12 floats (normal, 3 vertices) + uint16
static int parse_binary(const unsigned char *b, size_t len, float **tri, int64_t *ntri) {
    if (len < 84) return SDF_EIO;
    uint32_t n;
    memcpy(&n, b + 80, 4);
    if ((size_t)84 + (size_t)50 * n != len || n == 0) return SDF_EIO;
    float *t = (float *)malloc(sizeof(float) * 9 * (size_t)n);
    if (!t) return SDF_ENOMEM;
    for (uint32_t i = 0; i < n; i++) memcpy(t + 9 * (size_t)i, b + 84 + 50 * (size_t)i + 12, 36);
    *tri = t; *ntri = n;
    return SDF_OK;
}

// ASCII: tokens; every "vertex x y z" is a corner, three per facet
static int parse_ascii(const char *s, float **tri, int64_t *ntri) {
    size_t cap = 1024, nv = 0;
    float *t = (float *)malloc(sizeof(float) * 3 * cap);
    if (!t) return SDF_ENOMEM;
    const char *p = s;
    int in_loop = 0, corners = 0, status = SDF_OK;
    while (*p) {
        while (*p && isspace((unsigned char)*p)) p++;
        const char *w = p;
        while (*p && !isspace((unsigned char)*p)) p++;
        const size_t wl = (size_t)(p - w);
        if (wl == 6 && !strncmp(w, "vertex", 6)) {
            if (!in_loop || corners >= 3) { status = SDF_EIO; break; }
            if (nv == cap) {
                cap *= 2;
                float *t2 = (float *)realloc(t, sizeof(float) * 3 * cap);
                if (!t2) { status = SDF_ENOMEM; break; }
                t = t2;
            }
            for (int k = 0; k < 3; k++) {
                char *end;
                t[3 * nv + k] = strtof(p, &end);
                if (end == p) { status = SDF_EIO; break; }
                p = end;
            }
            if (status != SDF_OK) break;
            nv++; corners++;
        } else if (wl == 5 && !strncmp(w, "outer", 5)) {
            in_loop = 1; corners = 0;
        } else if (wl == 7 && !strncmp(w, "endloop", 7)) {
            if (!in_loop || corners != 3) { status = SDF_EIO; break; }
            in_loop = 0;
        }
    }
    if (status == SDF_OK && (in_loop || nv == 0 || nv % 3 != 0)) status = SDF_EIO;
    if (status != SDF_OK) { free(t); return status; }
    *tri = t; *ntri = (int64_t)(nv / 3);
    return SDF_OK;
}

extern "C" {

int sdf_read_stl(const char *path, float **tri_xyz_out, int64_t *ntri_out) {
    if (tri_xyz_out) *tri_xyz_out = nullptr;
    if (ntri_out) *ntri_out = 0;
    if (!path || !tri_xyz_out || !ntri_out) return SDF_EINVAL;
    unsigned char *b = nullptr;
    size_t len = 0;
    CKS(read_all(path, &b, &len));
    // ASCII files start with "solid" and carry the word "facet"; a binary header may start with
    // "solid" too, so the exact binary size relation decides first
    int s = parse_binary(b, len, tri_xyz_out, ntri_out);
    if (s == SDF_EIO) {
        const char *c = (const char *)b;
        while (*c && isspace((unsigned char)*c)) c++;
        if (!strncmp(c, "solid", 5) && strstr(c, "facet")) s = parse_ascii(c, tri_xyz_out, ntri_out);
    }
    free(b);
    return s;
}

void sdf_free_host(void *p) { free(p); }

int sdf_write_stl(const char *path, const float *tri_xyz, int64_t ntri, int ascii) {
    if (!path || !tri_xyz || ntri <= 0 || ntri > 0xFFFFFFFFll) return SDF_EINVAL;
    FILE *f = fopen(path, "wb");
    if (!f) return SDF_EIO;
    int ok = 1;
    if (ascii) {
        ok &= fprintf(f, "solid sdf\n") > 0;
        for (int64_t i = 0; i < ntri && ok; i++) {
            const float *T = tri_xyz + 9 * i;
            const double u[3] = {(double)T[3] - T[0], (double)T[4] - T[1], (double)T[5] - T[2]};
            const double v[3] = {(double)T[6] - T[0], (double)T[7] - T[1], (double)T[8] - T[2]};
            double n[3] = {u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0]};
            const double L = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
            if (L > 0.0) { n[0] /= L; n[1] /= L; n[2] /= L; }
            ok &= fprintf(f, "facet normal %.9g %.9g %.9g\nouter loop\n", n[0], n[1], n[2]) > 0;
            for (int k = 0; k < 3; k++) ok &= fprintf(f, "vertex %.9g %.9g %.9g\n", T[3 * k], T[3 * k + 1], T[3 * k + 2]) > 0;
            ok &= fprintf(f, "endloop\nendfacet\n") > 0;
        }
        ok &= fprintf(f, "endsolid sdf\n") > 0;
    } else {
        unsigned char hdr[80];
        memset(hdr, 0, sizeof(hdr));
        memcpy(hdr, "binary stl written by sdf_write_stl", 35);
        const uint32_t n = (uint32_t)ntri;
        ok &= fwrite(hdr, 1, 80, f) == 80 && fwrite(&n, 4, 1, f) == 1;
        for (int64_t i = 0; i < ntri && ok; i++) {
            const float *T = tri_xyz + 9 * i;
            const double u[3] = {(double)T[3] - T[0], (double)T[4] - T[1], (double)T[5] - T[2]};
            const double v[3] = {(double)T[6] - T[0], (double)T[7] - T[1], (double)T[8] - T[2]};
            double n3[3] = {u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0]};
            const double L = sqrt(n3[0] * n3[0] + n3[1] * n3[1] + n3[2] * n3[2]);
            float rec[12];
            for (int k = 0; k < 3; k++) rec[k] = (float)(L > 0.0 ? n3[k] / L : 0.0);
            memcpy(rec + 3, T, 36);
            const uint16_t attr = 0;
            ok &= fwrite(rec, 4, 12, f) == 12 && fwrite(&attr, 2, 1, f) == 1;
        }
    }
    if (fclose(f) != 0) ok = 0;
    return ok ? SDF_OK : SDF_EIO;
}

// grid file (the paper does not give its layout: this one is the library's own): the 8 bytes
// "SDFGRID1", int32 nx, ny, nz, has_tri, float origin[3], h, band, then nx*ny*nz floats (x fastest)
// and, if has_tri, nx*ny*nz int32
int sdf_write_grid(const char *path, const float *dist_host, const int32_t *tri_host, const float origin[3], float h,
                   int nx, int ny, int nz, float band) {
    if (!path || !dist_host || !origin || nx <= 0 || ny <= 0 || nz <= 0) return SDF_EINVAL;
    FILE *f = fopen(path, "wb");
    if (!f) return SDF_EIO;
    const int32_t ih[4] = {nx, ny, nz, tri_host ? 1 : 0};
    const float fh[5] = {origin[0], origin[1], origin[2], h, band};
    const size_t n = (size_t)nx * ny * nz;
    int ok = fwrite("SDFGRID1", 1, 8, f) == 8 && fwrite(ih, 4, 4, f) == 4 && fwrite(fh, 4, 5, f) == 5;
    ok = ok && fwrite(dist_host, 4, n, f) == n;
    if (ok && tri_host) ok = fwrite(tri_host, 4, n, f) == n;
    if (fclose(f) != 0) ok = 0;
    return ok ? SDF_OK : SDF_EIO;
}

} // extern "C"
