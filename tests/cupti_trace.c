/* Test infrastructure (not product code): counts CUDA runtime API calls by name between trace_begin() and
 * trace_end(), through CUPTI's callback API.  The automated form of the paper's "visual inspection of the timeline"
 * for the property PAPER.md:41 step 5 and :71 are about: nothing inside aa_run allocates, frees or
 * synchronises the device.  Built by tests/test_gpu_api_trace.py with gcc against the toolkit's libcupti. */
#include <cupti.h>
#include <pthread.h>
#include <stdio.h>
#include <string.h>

#define MAXN 128
static CUpti_SubscriberHandle g_sub;
static pthread_mutex_t g_mu = PTHREAD_MUTEX_INITIALIZER;
static char g_name[MAXN][64];
static long g_count[MAXN];
static int g_n, g_on;

static void CUPTIAPI on_call(void *ud, CUpti_CallbackDomain dom, CUpti_CallbackId cbid, const void *cbdata)
{
    (void)ud; (void)cbid;
    if (dom != CUPTI_CB_DOMAIN_RUNTIME_API) return;
    const CUpti_CallbackData *d = (const CUpti_CallbackData *)cbdata;
    if (d->callbackSite != CUPTI_API_ENTER || !d->functionName) return;
    pthread_mutex_lock(&g_mu);
    int i;
    for (i = 0; i < g_n; ++i)
        if (!strncmp(g_name[i], d->functionName, 63)) break;
    if (i == g_n && g_n < MAXN) {
        strncpy(g_name[g_n], d->functionName, 63);
        g_name[g_n][63] = 0;
        g_count[g_n++] = 0;
    }
    if (i < MAXN) g_count[i]++;
    pthread_mutex_unlock(&g_mu);
}

/* 0 on success, else the CUptiResult */
int trace_begin(void)
{
    g_n = 0;
    CUptiResult r = cuptiSubscribe(&g_sub, (CUpti_CallbackFunc)on_call, NULL);
    if (r != CUPTI_SUCCESS) return (int)r;
    r = cuptiEnableDomain(1, g_sub, CUPTI_CB_DOMAIN_RUNTIME_API);
    if (r != CUPTI_SUCCESS) { cuptiUnsubscribe(g_sub); return (int)r; }
    g_on = 1;
    return 0;
}

/* writes "name count\n" lines into buf; returns the number of distinct runtime functions seen */
int trace_end(char *buf, int len)
{
    if (g_on) { cuptiUnsubscribe(g_sub); g_on = 0; }
    int pos = 0;
    for (int i = 0; i < g_n && pos < len - 96; ++i) pos += snprintf(buf + pos, (size_t)(len - pos), "%s %ld\n", g_name[i], g_count[i]);
    if (len > 0) buf[pos < len ? pos : len - 1] = 0;
    return g_n;
}
