/*
 * vr_vmm.cu -- a brick store that can be handed back brick by brick (CUDA virtual memory management).
 *
 * Why: the texture arm of rows a1 / a5 (vr_texture.cu) keeps the bricks a second time, as 3-D CUDA
 * arrays, and two copies of the 103 GB cube do not fit 180 GB. A store made of one physical allocation per brick, mapped
 * into ONE contiguous virtual range, lets vr_volume_release_store fill a brick's array and give the brick's float32
 * cells back before the next array is allocated (peak: the store plus one array) - without any kernel noticing: the
 * store stays `base + slot * slot_bytes` for everything that is still mapped.
 *
 * Layout: chunk s covers the bytes [B_s, B_{s+1}) of the range, B_s = floor(s * slot_bytes / G) * G for the allocation
 * granularity G (2 MB), B_n = the rounded-up total. Slot s therefore lives in chunks s and s + 1 (its last < G bytes), and
 * chunk s can be released once slots s - 1 and s are both released.
 *
 * The driver entry points come from cudaGetDriverEntryPoint (libvr links the runtime only).
 */
#include <cuda.h>
#include <string.h>

#include <new>

#include "vr_internal.cuh"

struct VrVmm {
    CUdeviceptr base;
    size_t total;      /* bytes reserved (a multiple of the granularity) */
    size_t slot_bytes;
    int nslots;
    size_t gran;
    CUmemGenericAllocationHandle* chunk; /* nslots handles (chunk s = [bound[s], bound[s+1])); 0 once released */
    size_t* bound;                       /* nslots + 1 */
    unsigned char* slot_released;        /* nslots */
};

struct VmmApi {
    CUresult (*GetGranularity)(size_t*, const CUmemAllocationProp*, CUmemAllocationGranularity_flags);
    CUresult (*AddressReserve)(CUdeviceptr*, size_t, size_t, CUdeviceptr, unsigned long long);
    CUresult (*AddressFree)(CUdeviceptr, size_t);
    CUresult (*Create)(CUmemGenericAllocationHandle*, size_t, const CUmemAllocationProp*, unsigned long long);
    CUresult (*Release)(CUmemGenericAllocationHandle);
    CUresult (*Map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long);
    CUresult (*Unmap)(CUdeviceptr, size_t);
    CUresult (*SetAccess)(CUdeviceptr, size_t, const CUmemAccessDesc*, size_t);
    bool ok;
};

static const VmmApi* vmm_api() {
    static VmmApi api;
    static bool looked = false;
    if (!looked) {
        looked = true;
        memset(&api, 0, sizeof(api));
        struct {
            const char* name;
            void** slot;
        } syms[] = {{"cuMemGetAllocationGranularity", (void**)&api.GetGranularity}, {"cuMemAddressReserve", (void**)&api.AddressReserve},
                    {"cuMemAddressFree", (void**)&api.AddressFree},                 {"cuMemCreate", (void**)&api.Create},
                    {"cuMemRelease", (void**)&api.Release},                         {"cuMemMap", (void**)&api.Map},
                    {"cuMemUnmap", (void**)&api.Unmap},                             {"cuMemSetAccess", (void**)&api.SetAccess}};
        api.ok = true;
        for (auto& s : syms) {
            cudaDriverEntryPointQueryResult qr;
            if (cudaGetDriverEntryPoint(s.name, s.slot, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !*s.slot)
                api.ok = false;
        }
        cudaGetLastError();
    }
    return &api;
}

void vr_vmm_destroy(VrVmm* m) {
    if (!m) return;
    const VmmApi* a = vmm_api();
    if (a->ok && m->base) {
        for (int s = 0; s < m->nslots; ++s)
            if (m->chunk && m->chunk[s]) {
                a->Unmap(m->base + m->bound[s], m->bound[s + 1] - m->bound[s]);
                a->Release(m->chunk[s]);
            }
        a->AddressFree(m->base, m->total);
    }
    delete[] m->chunk;
    delete[] m->bound;
    delete[] m->slot_released;
    delete m;
}

/* cudaErrorNotSupported: no VMM on this driver / device; cudaErrorMemoryAllocation: out of memory */
cudaError_t vr_vmm_create(size_t slot_bytes, int nslots, VrVmm** out, float** base_out) {
    *out = NULL;
    *base_out = NULL;
    const VmmApi* a = vmm_api();
    if (!a->ok) return cudaErrorNotSupported;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return cudaErrorNotSupported;
    cudaFree(0); /* make sure the primary context exists */
    CUmemAllocationProp prop;
    memset(&prop, 0, sizeof(prop));
    prop.type = CU_MEM_ALLOCATION_TYPE_PINNED;
    prop.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    prop.location.id = dev;
    size_t gran = 0;
    if (a->GetGranularity(&gran, &prop, CU_MEM_ALLOC_GRANULARITY_MINIMUM) != CUDA_SUCCESS || gran == 0) return cudaErrorNotSupported;
    VrVmm* m = new (std::nothrow) VrVmm();
    if (!m) return cudaErrorMemoryAllocation;
    memset(m, 0, sizeof(*m));
    m->slot_bytes = slot_bytes;
    m->nslots = nslots;
    m->gran = gran;
    m->total = ((slot_bytes * (size_t)nslots + gran - 1) / gran) * gran;
    m->chunk = new (std::nothrow) CUmemGenericAllocationHandle[nslots]();
    m->bound = new (std::nothrow) size_t[nslots + 1];
    m->slot_released = new (std::nothrow) unsigned char[nslots]();
    if (!m->chunk || !m->bound || !m->slot_released) {
        vr_vmm_destroy(m);
        return cudaErrorMemoryAllocation;
    }
    for (int s = 0; s < nslots; ++s) m->bound[s] = ((slot_bytes * (size_t)s) / gran) * gran;
    m->bound[nslots] = m->total;
    if (a->AddressReserve(&m->base, m->total, 0, 0, 0) != CUDA_SUCCESS) {
        m->base = 0;
        vr_vmm_destroy(m);
        return cudaErrorMemoryAllocation;
    }
    CUmemAccessDesc acc;
    memset(&acc, 0, sizeof(acc));
    acc.location = prop.location;
    acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
    for (int s = 0; s < nslots; ++s) {
        const size_t len = m->bound[s + 1] - m->bound[s];
        if (len == 0) continue; /* slots smaller than the granularity share a chunk with their neighbour */
        CUresult r = a->Create(&m->chunk[s], len, &prop, 0);
        if (r == CUDA_SUCCESS) {
            r = a->Map(m->base + m->bound[s], len, 0, m->chunk[s], 0);
            if (r != CUDA_SUCCESS) {
                a->Release(m->chunk[s]);
                m->chunk[s] = 0;
            }
        } else {
            m->chunk[s] = 0;
        }
        if (r == CUDA_SUCCESS) r = a->SetAccess(m->base + m->bound[s], len, &acc, 1);
        if (r != CUDA_SUCCESS) {
            vr_vmm_destroy(m);
            return r == CUDA_ERROR_OUT_OF_MEMORY ? cudaErrorMemoryAllocation : cudaErrorUnknown;
        }
    }
    *out = m;
    *base_out = reinterpret_cast<float*>(m->base);
    return cudaSuccess;
}

/* Slot s is no longer needed: release every chunk whose slots are all released. Returns the bytes given back.
 * The caller has synchronised: no kernel is reading the slot. */
size_t vr_vmm_release_slot(VrVmm* m, int s) {
    const VmmApi* a = vmm_api();
    if (!m || s < 0 || s >= m->nslots || m->slot_released[s]) return 0;
    m->slot_released[s] = 1;
    size_t freed = 0;
    for (int c = s; c <= s + 1 && c < m->nslots; ++c) {
        if (!m->chunk[c]) continue;
        /* chunk c holds bytes of the slots that overlap [bound[c], bound[c+1]) */
        const size_t lo = m->bound[c], hi = m->bound[c + 1];
        bool all = true;
        for (int t = (int)(lo / m->slot_bytes); t < m->nslots && (size_t)t * m->slot_bytes < hi; ++t)
            if (!m->slot_released[t]) all = false;
        if (!all) continue;
        a->Unmap(m->base + lo, hi - lo);
        a->Release(m->chunk[c]);
        m->chunk[c] = 0;
        freed += hi - lo;
    }
    return freed;
}

int vr_vmm_slot_released(const VrVmm* m, int s) { return m && s >= 0 && s < m->nslots ? m->slot_released[s] : 0; }
